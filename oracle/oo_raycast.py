"""CPU ORACLE (numpy, float64) for the step BEFORE the query: primary visibility of the analytic stand-in scene
("rendering reduces to standard primary visibility plus one
OctaOctree query and one decoder evaluation per visible shading point").

TEST INFRASTRUCTURE ONLY (same rules as oo_oracle.py).  It shares nothing with the CUDA path (oo_raycast.cu) nor with the
input generator's C ray caster (gen/oo_gen.c), against which tests/test_oracle_raycast.py cross-checks it.

The paper traces its G-buffers with Mitsuba 3, which is not available here; the scene is BASELINE.json's
"analytic scene of spheres plus a 5-plane box in the unit cube".  What is computed, written out:

  camera   pinhole: f = normalize(look - eye), r = normalize(f x up), u = r x f, th = tan(vfov/2), aspect = W/H;
           pixel (i, j), centre sampled: px = (2 (i + 1/2)/W - 1) th aspect, py = (1 - 2 (j + 1/2)/H) th,
           d = normalize(f + px r + py u); rays leave the eye; scanline order q = j W + i.
  sphere   (c, R): oc = o - c, b = oc . d, cc = oc . oc - R^2, disc = b^2 - cc; no hit if disc < 0;
           t = -b - sqrt(disc), or -b + sqrt(disc) if that is <= tmin (the eye inside the sphere).
  plane    axis a at position p, a rectangle [lo, hi]^2 on the other two axes: t = (p - o_a)/d_a; hit if the other two
           coordinates of o + t d lie in [lo, hi].
  nearest  the smallest t > tmin = 1e-9 over the spheres in order, then the planes in order (x=lo, x=hi, y=lo, y=hi,
           z=lo); a later surface replaces an earlier one only if its t is strictly smaller.
  outputs  x = o + t d, n = (x - c)/R for a sphere (outward) or the unit axis vector pointing into the box for a plane,
           wo = -d, each rounded once to fp32; surface id (spheres 0..S-1, planes S..S+4), -1 and zeros for a miss.
Dot products and norms are summed left to right; nothing is fused.
"""
from __future__ import annotations

import numpy as np

PLANE_AXIS = (0, 0, 1, 1, 2)
PLANE_SIDE = (0, 1, 0, 1, 0)      # 0: at lo, 1: at hi
TMIN = 1e-9


def _dot(a, b):
    return (a[..., 0] * b[..., 0] + a[..., 1] * b[..., 1]) + a[..., 2] * b[..., 2]


def _normalize(v):
    return v / np.sqrt(_dot(v, v))[..., None]


def _cross(a, b):
    return np.stack([a[..., 1] * b[..., 2] - a[..., 2] * b[..., 1], a[..., 2] * b[..., 0] - a[..., 0] * b[..., 2],
                     a[..., 0] * b[..., 1] - a[..., 1] * b[..., 0]], -1)


def camera_basis(eye, look, up, vfov_deg):
    eye, look, up = (np.asarray(v, np.float64) for v in (eye, look, up))
    f = _normalize(look - eye)
    r = _normalize(_cross(f, up))
    u = _cross(r, f)
    th = np.tan(0.5 * vfov_deg * 3.14159265358979323846 / 180.0)
    return f, r, u, float(th)


def primary_rays(eye, look, up, vfov_deg, width, height, rows=None):
    """Unit directions [n_rows*W][3] of the pixel-centre rays, scanline order."""
    f, r, u, th = camera_basis(eye, look, up, vfov_deg)
    aspect = float(width) / float(height)
    rows = np.arange(height) if rows is None else np.asarray(rows)
    i = np.arange(width, dtype=np.float64)[None, :]
    j = rows.astype(np.float64)[:, None]
    px = np.broadcast_to((2.0 * (i + 0.5) / width - 1.0) * th * aspect, (len(rows), width)).reshape(-1)
    py = np.broadcast_to((1.0 - 2.0 * (j + 0.5) / height) * th, (len(rows), width)).reshape(-1)
    d = (f[None, :] + px[:, None] * r[None, :]) + py[:, None] * u[None, :]
    return _normalize(d)


def scene_hit(spheres, lo, hi, o, d):
    """Nearest hit of rays o + t d.  Returns t [N] (inf = miss), surface id [N] (-1 = miss)."""
    spheres = np.asarray(spheres, np.float64).reshape(-1, 4)
    o = np.asarray(o, np.float64)
    N = d.shape[0]
    best = np.full(N, np.inf)
    surf = np.full(N, -1, np.int64)
    for s, sp in enumerate(spheres):
        oc = o - sp[:3]
        b = _dot(np.broadcast_to(oc, d.shape), d)
        cc = _dot(oc, oc) - sp[3] * sp[3]
        disc = b * b - cc
        ok = disc >= 0.0
        sq = np.sqrt(np.where(ok, disc, 0.0))
        t = -b - sq
        t = np.where(t <= TMIN, -b + sq, t)
        take = ok & (t > TMIN) & (t < best)
        best = np.where(take, t, best)
        surf = np.where(take, s, surf)
    for p in range(5):
        ax = PLANE_AXIS[p]
        pos = hi if PLANE_SIDE[p] else lo
        nz = d[:, ax] != 0.0
        t = (pos - o[ax]) / np.where(nz, d[:, ax], 1.0)
        take = nz & (t > TMIN) & (t < best)
        for a in range(3):
            if a != ax:
                q = o[a] + t * d[:, a]
                take &= (q >= lo) & (q <= hi)
        best = np.where(take, t, best)
        surf = np.where(take, len(spheres) + p, surf)
    return best, surf


def raycast(spheres, lo, hi, eye, look, up, vfov_deg, width, height, rows=None):
    """The primary-hit queries of a frame: x, n, wo as fp32 [N][3] and the surface id [N]."""
    spheres = np.asarray(spheres, np.float64).reshape(-1, 4)
    o = np.asarray(eye, np.float64)
    d = primary_rays(eye, look, up, vfov_deg, width, height, rows)
    t, surf = scene_hit(spheres, lo, hi, o, d)
    hit = surf >= 0
    ts = np.where(hit, t, 0.0)
    x = o[None, :] + ts[:, None] * d
    n = np.zeros_like(x)
    S = len(spheres)
    is_sph = hit & (surf < S)
    if S:
        sp = spheres[np.clip(surf, 0, S - 1)]
        n = np.where(is_sph[:, None], (x - sp[:, :3]) / sp[:, 3:4], n)
    for p in range(5):
        m = surf == S + p
        n[m, PLANE_AXIS[p]] = -1.0 if PLANE_SIDE[p] else 1.0
    x = np.where(hit[:, None], x, 0.0)
    wo = np.where(hit[:, None], -d, 0.0)
    return x.astype(np.float32), n.astype(np.float32), wo.astype(np.float32), surf
