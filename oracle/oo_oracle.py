"""CPU ORACLE (numpy, float64) for the OctaOctree per-query radiance evaluation.

TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, obviously-correct restatement of what the
hot path computes, written from the paper (/root/reference/PAPER.md, cited as P:line) and from the
readings of it listed in DESIGN.md ("Readings", A1-A24).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import it.  It shares no code, table, constant
or helper with the CUDA path (paper_2606_08469_b200/) and imports nothing from it; inputs are
passed in as plain numpy arrays.

Everything is double precision, EXCEPT the one integer decision that floating point takes: the
base texel (i0, j0) of the bilinear footprint, which both sides take in fp32 with the fixed
operation sequence of `texel_base_f32`.  Weights and sums stay double.

What is computed, per query (x, n, wo[, extra]) ("one OctaOctree query and one decoder
evaluation per visible shading point"):

  O1 quantise   q_a = clamp(floor(x_a * 2^Dmax), 0, 2^Dmax-1)                  cells of P:160-164
  O2 descent    follow child[node][octant] from the root; slot per used level  sparse octree, P:160
  O3 octa map   u = (wx, wy)/(|wx|+|wy|+|wz|); fold if wz<0                    Eq. 4-5
  O4 remap      v = (u+1)/2 in [0,1]^2; s = v*R - 1/2 (texel centres)          P:121 (+ A2, A3)
  O5 wrap       out-of-range taps continue on the neighbouring octahedron face P:125 ("continuous
                across the spherical domain")
  O6 interpolate 4-tap bilinear, the nearest-cell / texel variant of Eq. 6/10
  O7 concat     [h_0 .. h_{L-1} | n | wo | extra]                              Eq. 11-13
  O8 decoder    H x (linear, ReLU), linear, exp                                f_phi

Pins (tests/test_oracle_*.py): see DESIGN.md "Oracle pins".  No end-to-end golden RGB exists in the
paper, so absolute end-to-end output is pinned by composition only (each step pinned separately,
plus closed-form end-to-end cases and an independent second implementation, oracle/oo_oracle.c).
"""
from __future__ import annotations

import numpy as np

# ------------------------------------------------------------------------------------------ O1, O2


def quantise(x, max_depth):
    """O1. Integer cell coordinates at the finest depth: q = clamp(floor(x * 2^Dmax), 0, 2^Dmax - 1).

    "For a query point x ... octree cells at level l".  Half-open cells [k, k+1)/2^d; x outside
    the unit cube is clamped componentwise (A15, A16).  Multiplying by a power of two is exact, so the
    result does not depend on whether x is held in fp32 or fp64."""
    x = np.asarray(x, np.float64)
    n_cells = 1 << max_depth
    q = np.floor(x * float(n_cells))
    return np.clip(q, 0, n_cells - 1).astype(np.int64)


def descend(child, q, max_depth):
    """O2. path[:, d] = id of the node of depth d that contains the query, or -1 once a child is absent.

    Octant at depth d (1-based step): bit (Dmax - d) of each coordinate, o = bx | by<<1 | bz<<2.
    "Each level partitions scene space into sparse octree cells"."""
    child = np.asarray(child)
    n = q.shape[0]
    path = np.full((n, max_depth + 1), -1, np.int64)
    node = np.zeros(n, np.int64)
    alive = np.ones(n, bool)
    path[:, 0] = 0
    for d in range(1, max_depth + 1):
        s = max_depth - d
        o = ((q[:, 0] >> s) & 1) | (((q[:, 1] >> s) & 1) << 1) | (((q[:, 2] >> s) & 1) << 2)
        nxt = np.where(alive, child[np.where(alive, node, 0), o], -1)
        alive = alive & (nxt >= 0)
        node = np.where(alive, nxt, node)
        path[:, d] = np.where(alive, nxt, -1)
    return path


def slots_from_path(path, map_slot, level_depth):
    """slot[:, l] = map_slot[node at depth d_l], -1 if that node is absent (A17: the level then contributes zeros)."""
    map_slot = np.asarray(map_slot)
    out = np.full((path.shape[0], len(level_depth)), -1, np.int64)
    for l, d in enumerate(level_depth):
        node = path[:, d]
        ok = node >= 0
        out[ok, l] = map_slot[node[ok]]
    return out


# ---------------------------------------------------------------------------------------------- O3


def _sgn(t):
    """sign with sign(0) = +1 (A1): with sign(0) = 0, -z would collide with +z at u = (0, 0)."""
    return np.where(t >= 0, 1.0, -1.0)


def octa_encode(w):
    """O3. Eq. 4: u = (wx, wy) / (|wx|+|wy|+|wz|); Eq. 5: if wz < 0, u <- ((1-|uy|) sgn ux, (1-|ux|) sgn uy)."""
    w = np.asarray(w, np.float64)
    S = np.abs(w[..., 0]) + np.abs(w[..., 1]) + np.abs(w[..., 2])
    ux, uy = w[..., 0] / S, w[..., 1] / S
    fx, fy = (1.0 - np.abs(uy)) * _sgn(ux), (1.0 - np.abs(ux)) * _sgn(uy)
    lower = w[..., 2] < 0
    return np.stack([np.where(lower, fx, ux), np.where(lower, fy, uy)], -1)


def octa_decode(u):
    """Inverse of octa_encode on the unit sphere (used by the pins only): z = 1-|ux|-|uy|; unfold if z<0; normalise."""
    u = np.asarray(u, np.float64)
    ux, uy = u[..., 0], u[..., 1]
    z = 1.0 - np.abs(ux) - np.abs(uy)
    x = np.where(z < 0, (1.0 - np.abs(uy)) * _sgn(ux), ux)
    y = np.where(z < 0, (1.0 - np.abs(ux)) * _sgn(uy), uy)
    w = np.stack([x, y, z], -1)
    return w / np.linalg.norm(w, axis=-1, keepdims=True)


# ------------------------------------------------------------------------------------------ O4, O5


def sample_coord(u, R):
    """O4. "remapped to [0,1]^2": v = (u+1)/2; texel centres at (i+1/2)/R, so s = v*R - 1/2 (A2, A3)."""
    return (np.asarray(u, np.float64) + 1.0) / 2.0 * R - 0.5


def texel_base_f32(wo, R):
    """The index decision, in fp32, round-to-nearest, one operation at a time.

        S = (|wx| + |wy|) + |wz| ; ux = wx / S ; uy = wy / S
        if wz < 0: tx = 1 - |uy| ; ty = 1 - |ux| ; ux' = (ux >= 0 ? tx : -tx) ; uy' = (uy >= 0 ? ty : -ty)
        sx = ux * (R/2) + (R/2 - 1/2)       (the product is exact: R/2 is a power of two)
        i0 = floor(sx), j0 = floor(sy)      in [-1, R-1]
    Returns int64 arrays (i0, j0)."""
    f = np.float32
    w = np.asarray(wo, np.float32)
    wx, wy, wz = w[..., 0], w[..., 1], w[..., 2]
    S = (np.abs(wx) + np.abs(wy)) + np.abs(wz)
    ux, uy = wx / S, wy / S
    tx, ty = f(1) - np.abs(uy), f(1) - np.abs(ux)
    lower = wz < 0
    fx = np.where(lower, np.where(ux >= 0, tx, -tx), ux).astype(f)
    fy = np.where(lower, np.where(uy >= 0, ty, -ty), uy).astype(f)
    half_r, off = f(R / 2.0), f(R / 2.0 - 0.5)
    sx, sy = (fx * half_r).astype(f) + off, (fy * half_r).astype(f) + off
    assert sx.dtype == np.float32 and sy.dtype == np.float32
    return np.floor(sx).astype(np.int64), np.floor(sy).astype(np.int64)


def texel_base_f64(wo, R):
    """Same decision taken in double (statistics only: how often fp32 and fp64 pick a different base texel)."""
    s = sample_coord(octa_encode(np.asarray(wo, np.float32).astype(np.float64)), R)
    return np.floor(s[..., 0]).astype(np.int64), np.floor(s[..., 1]).astype(np.int64)


def wrap(i, j, R):
    """O5. A tap outside [0,R)^2 lies across an edge of the unfolded octahedron; the surface continues on the
    neighbouring face, which in the unfolded square is the point reflection about the midpoint of the crossed edge:
    (R, j) -> (R-1, R-1-j), (-1, j) -> (0, R-1-j), (i, R) -> (R-1-i, R-1), (i, -1) -> (R-1-i, 0)."""
    i, j = np.asarray(i).copy(), np.asarray(j).copy()
    out_i = (i < 0) | (i >= R)
    j = np.where(out_i, R - 1 - j, j)
    i = np.clip(i, 0, R - 1)
    out_j = (j < 0) | (j >= R)
    i = np.where(out_j, R - 1 - i, i)
    j = np.clip(j, 0, R - 1)
    return i, j


# ---------------------------------------------------------------------------------------------- O6


def dir_interp(T, slot, wo, R):
    """O6. h = sum over the four taps of (bilinear weight) x T[slot][j][i][:]; zeros where slot < 0.

    T: [slots][R][R][F] (any float dtype, widened exactly to double). The directional analogue of Eq. 6
    on a texel-centred map (A3, A4), inside the single cell that contains x (the nearest-cell variant)."""
    T = np.asarray(T)
    wo32 = np.asarray(wo, np.float32)
    i0, j0 = texel_base_f32(wo32, R)
    s = sample_coord(octa_encode(wo32.astype(np.float64)), R)
    fx, fy = s[..., 0] - i0, s[..., 1] - j0          # not clamped: continuous interpolant
    ok = slot >= 0
    sl = np.where(ok, slot, 0)
    h = np.zeros((wo32.shape[0], T.shape[-1]), np.float64)
    for b in (0, 1):
        for a in (0, 1):
            wgt = (fx if a else 1.0 - fx) * (fy if b else 1.0 - fy)
            ii, jj = wrap(i0 + a, j0 + b, R)
            h += wgt[:, None] * T[sl, jj, ii, :].astype(np.float64)
    h[~ok] = 0.0
    return h, i0, j0


# ------------------------------------------------------------------------------------------ O7, O8


def encode(tree, atlas_levels, x, wo):
    """O1-O6 and the feature part of O7: features [N][L*F] (levels coarse -> fine, Eq. 11), slots [N][L],
    base texels [N][L][2] = (i0, j0) before wrapping."""
    q = quantise(x, tree.max_depth)
    path = descend(tree.child, q, tree.max_depth)
    slots = slots_from_path(path, tree.map_slot, tree.level_depth)
    feats, tex = [], []
    for l, R in enumerate(tree.level_res):
        h, i0, j0 = dir_interp(atlas_levels[l], slots[:, l], wo, R)
        feats.append(h)
        tex.append(np.stack([i0, j0], -1))
    return np.concatenate(feats, 1), slots, np.stack(tex, 1)


def mlp_input(features, nrm, wo, extra=None):
    """O7. [h | n | wo | extra] (Eq. 11-13 with BASELINE.json's reduced g; A7). Raw values, no further encoding."""
    parts = [features, np.asarray(nrm, np.float32).astype(np.float64), np.asarray(wo, np.float32).astype(np.float64)]
    if extra is not None:
        parts.append(np.asarray(extra, np.float32).astype(np.float64).reshape(features.shape[0], -1))
    return np.concatenate(parts, 1)


def mlp(weights, inp, out_act="exp"):
    """O8. a <- max(W_k a, 0) for the hidden layers, z = W_H a, rgb = exp(z) (A9-A11; no biases)."""
    a = np.asarray(inp, np.float64)
    for W in weights[:-1]:
        a = np.maximum(a @ np.asarray(W).astype(np.float64).T, 0.0)
    z = a @ np.asarray(weights[-1]).astype(np.float64).T
    if out_act == "exp":
        return np.exp(z)
    if out_act == "none":
        return z
    raise ValueError(out_act)


def query(tree, atlas_levels, mlp_weights, x, nrm, wo, extra=None, out_act="exp"):
    """The whole path: rgb [N][3] in double."""
    feats, _, _ = encode(tree, atlas_levels, x, wo)
    return mlp(mlp_weights, mlp_input(feats, nrm, wo, extra), out_act)


# ------------------------------------------------------------------------------- Morton order (a1)


def morton_keys(x, bits=10):
    """30-bit Morton key of floor(x * 2^bits) clamped (row a1; not in the paper, BASELINE.json north_star):
    bit k of qx -> key bit 3k, qy -> 3k+1, qz -> 3k+2 (the same octant convention as the tree)."""
    q = quantise(x, bits)
    key = np.zeros(q.shape[0], np.int64)
    for k in range(bits):
        key |= ((q[:, 0] >> k) & 1) << (3 * k)
        key |= ((q[:, 1] >> k) & 1) << (3 * k + 1)
        key |= ((q[:, 2] >> k) & 1) << (3 * k + 2)
    return key


def morton_order(x, bits=10):
    """Stable argsort of the Morton keys (ties keep the original order): the unique expected permutation."""
    return np.argsort(morton_keys(x, bits), kind="stable")
