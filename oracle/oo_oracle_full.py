"""CPU ORACLE (numpy, float64) for the paper's FULL OctaOctree query — the NEXT rows of SURVEY.md §8(f).

TEST INFRASTRUCTURE ONLY (same rules as oo_oracle.py: only tests/, smoke() and bench.py's CPU legs import it; it shares
nothing with the CUDA path).  It widens the nearest-cell / texel / raw-wo hot path of oo_oracle.py to what the paper
describes (/root/reference/PAPER.md cited as P:line; readings in DESIGN.md §2 and §12):

  f1  spatial blend over the eight neighbouring cells with trilinear weights, non-empty indicator and
      renormalisation                                                              Eq. 10, P:164-168 (A5, A6)
  f2  directional features stored at the VERTICES of the unfolded octahedral grid, barycentric interpolation over the
      containing right-isosceles triangle, 3 taps                                  Eq. 6
  f3  lookup direction: mirror reflection direction w_r, optionally shifted per cell by a disparity d^:
      w~_j = normalize((x - c_j) d^ + w_r)                                          P:135, Eq. 8-9
      (d^ itself comes from the network g_psi of Eq. 7; it enters here as a per-query INPUT, or from
      oracle/oo_hashgrid.py when the disparity network is used)
  f4  attribute vector g = [x, w_r, n, extras] (extras = albedo a, roughness alpha)   Eq. 12

Every function follows the paper's order; `mode` selects the variant per piece so that the all-default mode
reproduces oo_oracle.py exactly (tests pin that).  Double precision throughout EXCEPT the decisions both sides take in
the kernel's precision: the base texel / grid cell of the directional lookup, the triangle
choice of f2, and — because every later index depends on it — the lookup direction itself (w_r and w~_j are formed in
fp32 by the fixed operation sequence of `mirror_f32` / `shifted_f32`, then widened).  Spatial weights, directional
weights and sums are double.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import oo_oracle as O


@dataclass
class Mode:
    spatial: str = "nearest"       # "nearest" (P:266 ablation, the hot path) | "trilinear8" (Eq. 10)
    dirmap: str = "texel"          # "texel" (R x R texel centres, bilinear, border wrap) | "vertex" ((R+1)^2 vertices, Eq. 6)
    lookup: str = "wo"             # "wo" (P:262 ablation, the hot path) | "mirror" (w_r) | "shifted" (Eq. 9)
    attrs: str = "n_wo"            # "n_wo": [n | wo | extras] (BASELINE.json) | "paper": [x | w_r | n | extras] (Eq. 12)


# ------------------------------------------------------------------------------------------------ f3: directions


def mirror_f32(nrm, wo):
    """w_r = 2 (n . wo) n - wo, the mirror reflection of the outgoing direction about the normal, in fp32 with
    one rounding per operation and no contraction: dot = ((n0*w0) + (n1*w1)) + (n2*w2); s = 2*dot (exact);
    w_r[a] = (s*n[a]) - wo[a]."""
    f = np.float32
    n = np.asarray(nrm, f)
    w = np.asarray(wo, f)
    dot = (((n[..., 0] * w[..., 0]).astype(f) + (n[..., 1] * w[..., 1]).astype(f)).astype(f) + (n[..., 2] * w[..., 2]).astype(f)).astype(f)
    s = (f(2) * dot).astype(f)
    return np.stack([((s * n[..., a]).astype(f) - w[..., a]).astype(f) for a in range(3)], -1)


def mirror_f64(nrm, wo):
    n = np.asarray(nrm, np.float32).astype(np.float64)
    w = np.asarray(wo, np.float32).astype(np.float64)
    return 2.0 * np.sum(n * w, -1, keepdims=True) * n - w


def shifted_f32(x, centre, disparity, w_r):
    """Eq. 9 numerator in fp32, one rounding per operation: w~[a] = ((x[a] - c[a]) * d^) + w_r[a].  Not normalised: Eq. 4
    divides by the L1 norm, so the octahedral image of w~ and of w~/||w~||_2 are the same point (A22).  `centre` is exact
    in fp32 ((k + 1/2) / 2^d)."""
    f = np.float32
    x = np.asarray(x, f)
    c = np.asarray(centre, f)
    d = np.asarray(disparity, f)[..., None]
    dx = (x - c).astype(f)
    return ((dx * d).astype(f) + np.asarray(w_r, f)).astype(f)


def shifted_f64(x, centre, disparity, w_r):
    """Eq. 8-9 literally, in double: y = x + w_r / d^;  w~ = (y - c) / ||y - c||_2  (statistics and pins only)."""
    x = np.asarray(x, np.float64)
    y = x + np.asarray(w_r, np.float64) / np.asarray(disparity, np.float64)[..., None]
    v = y - np.asarray(centre, np.float64)
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


# ------------------------------------------------------------------------------------------------ f2: vertex maps


def vertex_cell_f32(w, n):
    """The index decision of the vertex-map lookup, in fp32 (one rounding per operation):
    u from Eq. 4-5 as in oo_oracle.texel_base_f32; g = u*(n/2) + n/2 (exact product); cell = min(floor(g), n-1);
    (a, b) = g - cell; quadrant sign from the cell index; triangle: same-sign quadrants use the anti-diagonal
    (upper = a + b >= 1), opposite-sign quadrants the main diagonal (upper = b > a).
    Returns ci, cj (int64) and tri (0 = the triangle containing local corner (0,0) or (1,0)...; see `vertex_taps`)."""
    f = np.float32
    w = np.asarray(w, np.float32)
    wx, wy, wz = w[..., 0], w[..., 1], w[..., 2]
    S = (np.abs(wx) + np.abs(wy)) + np.abs(wz)
    ux, uy = (wx / S).astype(f), (wy / S).astype(f)
    tx, ty = f(1) - np.abs(uy), f(1) - np.abs(ux)
    lower = wz < 0
    fx = np.where(lower, np.where(ux >= 0, tx, -tx), ux).astype(f)
    fy = np.where(lower, np.where(uy >= 0, ty, -ty), uy).astype(f)
    h = f(n / 2.0)
    gx, gy = (fx * h).astype(f) + h, (fy * h).astype(f) + h
    ci = np.minimum(np.floor(gx), n - 1).astype(np.int64)
    cj = np.minimum(np.floor(gy), n - 1).astype(np.int64)
    ci, cj = np.maximum(ci, 0), np.maximum(cj, 0)
    a, b = (gx - ci.astype(f)).astype(f), (gy - cj.astype(f)).astype(f)
    same = (ci >= n // 2) == (cj >= n // 2)
    upper = np.where(same, (a + b).astype(f) >= f(1), b > a)
    return ci, cj, upper.astype(np.int64)


def vertex_taps(ci, cj, upper, a, b, n):
    """Eq. 6: the three vertices of the containing triangle and their barycentric weights.  Local corners of cell
    (ci, cj): (0,0), (1,0), (0,1), (1,1); (a, b) in [0,1]^2 are the local coordinates.

    After unfolding, the uniformly subdivided octahedron faces become right isosceles triangles whose hypotenuses are
    parallel to the face edge |u_x| + |u_y| = 1: the anti-diagonal where u_x u_y > 0, the main diagonal where
    u_x u_y < 0.  Figure 3 is missing from the reference text; this orientation follows from the geometry and is pinned
    against an independent 3-D barycentric construction on the octahedron faces (tests/test_oracle_full.py).
      anti-diagonal, lower (a+b < 1): (0,0) 1-a-b ; (1,0) a ; (0,1) b
      anti-diagonal, upper          : (1,1) a+b-1 ; (0,1) 1-a ; (1,0) 1-b
      main diagonal, lower (a >= b) : (0,0) 1-a ; (1,0) a-b ; (1,1) b
      main diagonal, upper (b > a)  : (0,0) 1-b ; (0,1) b-a ; (1,1) a
    Returns (iv [.,3], jv [.,3], wgt [.,3])."""
    same = (ci >= n // 2) == (cj >= n // 2)
    up = upper.astype(bool)
    z, o = np.zeros_like(ci), np.ones_like(ci)
    di = np.where(same[..., None], np.where(up[..., None], np.stack([o, z, o], -1), np.stack([z, o, z], -1)),
                  np.where(up[..., None], np.stack([z, z, o], -1), np.stack([z, o, o], -1)))
    dj = np.where(same[..., None], np.where(up[..., None], np.stack([o, o, z], -1), np.stack([z, z, o], -1)),
                  np.where(up[..., None], np.stack([z, o, o], -1), np.stack([z, z, o], -1)))
    wg = np.where(same[..., None],
                  np.where(up[..., None], np.stack([a + b - 1, 1 - a, 1 - b], -1), np.stack([1 - a - b, a, b], -1)),
                  np.where(up[..., None], np.stack([1 - b, b - a, a], -1), np.stack([1 - a, a - b, b], -1)))
    return ci[..., None] + di, cj[..., None] + dj, wg


def dir_interp_vertex(T, slot, w32, n):
    """Eq. 6 on one cell's vertex map.  T: [slots][n+1][n+1][F]; w32: fp32 lookup directions; zeros where slot < 0."""
    T = np.asarray(T)
    w32 = np.asarray(w32, np.float32)
    ci, cj, upper = vertex_cell_f32(w32, n)
    u = O.octa_encode(w32.astype(np.float64))
    g = (u + 1.0) / 2.0 * n                               # "remapped to [0,1]^2", times the grid resolution
    a, b = g[..., 0] - ci, g[..., 1] - cj                 # not clamped: the interpolant is continuous
    iv, jv, wg = vertex_taps(ci, cj, upper, a, b, n)
    ok = slot >= 0
    sl = np.where(ok, slot, 0)
    h = np.zeros((w32.shape[0], T.shape[-1]), np.float64)
    for k in range(3):
        h += wg[:, k, None] * T[sl, jv[:, k], iv[:, k], :].astype(np.float64)
    h[~ok] = 0.0
    return h, ci, cj, upper


# ------------------------------------------------------------------------------------------------ f1: spatial blend


def cell_node(child, k, depth):
    """Node id at `depth` whose integer cell coordinates are k [N,3] (or -1: outside the grid, or absent).  The plain
    descent of oo_oracle.descend applied to the cell's own coordinates."""
    n_c = 1 << depth
    inside = np.all((k >= 0) & (k < n_c), -1)
    kk = np.where(inside[:, None], k, 0).astype(np.int64)
    path = O.descend(child, kk, depth)
    return np.where(inside, path[:, depth], -1)


def neighbours(x, depth):
    """Eq. 10's eight neighbouring cells and "standard trilinear weights": features sit at cell centres, so with
    p = x 2^d - 1/2 (x clamped to the unit cube, A16), base cell k0 = floor(p), t = p - k0, neighbour j = a | b<<1 | c<<2
    is cell k0 + (a, b, c) with weight prod(t or 1-t).  Returns k [N,8,3] int64 and w [N,8] double."""
    xc = np.clip(np.asarray(x, np.float32).astype(np.float64), 0.0, 1.0)
    p = xc * float(1 << depth) - 0.5
    k0 = np.floor(p)
    t = p - k0
    k0 = k0.astype(np.int64)
    ks, ws = [], []
    for j in range(8):
        o = np.array([j & 1, (j >> 1) & 1, (j >> 2) & 1])
        ks.append(k0 + o)
        ws.append(np.prod(np.where(o.astype(bool), t, 1.0 - t), -1))
    return np.stack(ks, 1), np.stack(ws, 1)


# ------------------------------------------------------------------------------------------------ the full encode


def lookup_direction(mode: Mode, x, nrm, wo, centre=None, disparity=None):
    """fp32 lookup direction for one cell per query (see module docstring)."""
    if mode.lookup == "wo":
        return np.asarray(wo, np.float32)
    w_r = mirror_f32(nrm, wo)
    if mode.lookup == "mirror":
        return w_r
    if mode.lookup == "shifted":
        return shifted_f32(x, centre, disparity, w_r)
    raise ValueError(mode.lookup)


def _dir_interp(mode: Mode, T, slot, w32, R):
    if mode.dirmap == "texel":
        h, _, _ = O.dir_interp(T, slot, w32, R)
        return h
    if mode.dirmap == "vertex":
        h, _, _, _ = dir_interp_vertex(T, slot, w32, R)
        return h
    raise ValueError(mode.dirmap)


def encode_full(tree, atlas_levels, x, nrm, wo, mode: Mode, disparity=None, return_debug: bool = False):
    """Features [N][L*F] (Eq. 11: levels coarse -> fine) under `mode`.  With return_debug also the per-level neighbour
    slots [N][L][8] (trilinear8) or [N][L][1] (nearest)."""
    x32 = np.asarray(x, np.float32)
    N = x32.shape[0]
    feats, dbg = [], []
    for l, (d, R) in enumerate(zip(tree.level_depth, tree.level_res)):
        T = atlas_levels[l]
        n_c = 1 << d
        if mode.spatial == "nearest":
            q = O.quantise(x32, d)                                             # the cell containing x at depth d
            node = cell_node(tree.child, q, d)
            slot = np.where(node >= 0, np.asarray(tree.map_slot)[np.maximum(node, 0)], -1)
            centre = ((q + 0.5) / n_c).astype(np.float32)
            w32 = lookup_direction(mode, x32, nrm, wo, centre, disparity)
            feats.append(_dir_interp(mode, T, slot, w32, R))
            dbg.append(slot[:, None])
        elif mode.spatial == "trilinear8":
            k, w = neighbours(x32, d)
            slots = np.full((N, 8), -1, np.int64)
            for j in range(8):
                node = cell_node(tree.child, k[:, j], d)
                slots[:, j] = np.where(node >= 0, np.asarray(tree.map_slot)[np.maximum(node, 0)], -1)
            ind = (slots >= 0).astype(np.float64)                              # 1(c_j): the cell is non-empty
            den = np.sum(ind * w, 1)                                           # sum_p 1(c_p) w_p   (A5)
            h = np.zeros((N, np.asarray(T).shape[-1]), np.float64)
            for j in range(8):
                centre = ((k[:, j] + 0.5) / n_c).astype(np.float32)
                w32 = lookup_direction(mode, x32, nrm, wo, centre, disparity)
                hj = _dir_interp(mode, T, slots[:, j], w32, R)
                wj = np.where(den > 0, ind[:, j] * w[:, j] / np.where(den > 0, den, 1.0), 0.0)
                h += wj[:, None] * hj
            feats.append(h)
            dbg.append(slots)
        else:
            raise ValueError(mode.spatial)
    f = np.concatenate(feats, 1)
    return (f, np.stack(dbg, 1)) if return_debug else f


def mlp_input_full(features, x, nrm, wo, extra, mode: Mode):
    """Eq. 12-13: the decoder input.  "n_wo": [h | n | wo | extras]; "paper": [h | x | w_r | n | extras] with
    extras = (albedo a, roughness alpha) supplied by the caller; w_r is the fp32 mirror direction of `mirror_f32`."""
    if mode.attrs == "n_wo":
        return O.mlp_input(features, nrm, wo, extra)
    if mode.attrs == "paper":
        w = lambda a: np.asarray(a, np.float32).astype(np.float64)
        parts = [features, w(x), w(mirror_f32(nrm, wo)), w(nrm)]
        if extra is not None:
            parts.append(w(extra).reshape(features.shape[0], -1))
        return np.concatenate(parts, 1)
    raise ValueError(mode.attrs)


def query_full(tree, atlas_levels, mlp_weights, x, nrm, wo, extra=None, out_act="exp", mode: Optional[Mode] = None,
               disparity=None):
    mode = mode or Mode()
    f = encode_full(tree, atlas_levels, x, nrm, wo, mode, disparity)
    return O.mlp(mlp_weights, mlp_input_full(f, x, nrm, wo, extra, mode), out_act)
