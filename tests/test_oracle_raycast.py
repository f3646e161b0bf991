"""Pins for oracle/oo_raycast.py (primary visibility of the analytic scene): closed forms,
implicit-surface invariants, brute-force ray marching, and the input generator's independent C ray caster."""
import numpy as np

import gen
from oracle import oo_raycast as RC

UP = (0.0, 1.0, 0.0)


def test_single_pixel_looks_along_the_view_axis_and_corner_rays_span_the_fov():
    d = RC.primary_rays((0.5, 0.5, 0.9), (0.5, 0.5, 0.1), UP, 60.0, 1, 1)
    assert np.allclose(d, [[0.0, 0.0, -1.0]], atol=1e-15)
    # 2x2 frame, square: pixel centres sit at half the half-extent, so tan(angle to the axis) = tan(30 deg)/2 * sqrt(2)
    d = RC.primary_rays((0.5, 0.5, 0.9), (0.5, 0.5, 0.1), UP, 60.0, 2, 2)
    ang = np.arccos(-d[:, 2])
    assert np.allclose(np.tan(ang), np.tan(np.radians(30.0)) / 2 * np.sqrt(2.0), atol=1e-14)
    # scanline order, image y down, x to the right (r = f x up = +x for a camera looking down -z with up = +y)
    assert d[0, 0] < 0 < d[1, 0] and d[0, 1] > 0 > d[2, 1]
    # aspect: a 4x2 frame's outermost columns are twice as far out as its outermost rows
    d = RC.primary_rays((0.5, 0.5, 0.9), (0.5, 0.5, 0.1), UP, 60.0, 4, 2)
    assert np.isclose((d[3, 0] / -d[3, 2]) / (d[0, 1] / -d[0, 2]), (0.75 * 2.0) / 0.5, atol=1e-13)
    assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-15)


def test_ray_through_a_sphere_centre_and_onto_the_back_plane():
    sph = np.array([[0.5, 0.5, 0.4, 0.1]])
    x, n, wo, s = RC.raycast(sph, 0.03, 0.97, (0.5, 0.5, 0.9), (0.5, 0.5, 0.1), UP, 60.0, 1, 1)
    assert s[0] == 0 and np.allclose(x[0], [0.5, 0.5, 0.5], atol=1e-7)          # |c - o| - R = 0.5 - 0.1 from z = 0.9
    assert np.allclose(n[0], [0, 0, 1], atol=1e-7) and np.allclose(wo[0], [0, 0, 1], atol=1e-7)
    x, n, wo, s = RC.raycast(np.zeros((0, 4)), 0.03, 0.97, (0.5, 0.5, 0.9), (0.5, 0.5, 0.1), UP, 60.0, 1, 1)
    assert s[0] == 4 and np.allclose(x[0], [0.5, 0.5, 0.03], atol=1e-7) and np.array_equal(n[0], [0, 0, 1])
    # eye inside a sphere: the far root
    t, s = RC.scene_hit(np.array([[0.5, 0.5, 0.9, 0.2]]), 0.03, 0.97, (0.5, 0.5, 0.9), np.array([[0.0, 0.0, -1.0]]))
    assert s[0] == 0 and np.isclose(t[0], 0.2, atol=1e-15)
    # a ray pointing out of the open side misses everything
    t, s = RC.scene_hit(np.zeros((0, 4)), 0.03, 0.97, (0.5, 0.5, 0.5), np.array([[0.0, 0.0, 1.0]]))
    assert s[0] == -1 and np.isinf(t[0])
    # side planes: normals point into the box
    for dvec, sid, nn in (((-1.0, 0, 0), 0, (1, 0, 0)), ((1.0, 0, 0), 1, (-1, 0, 0)), ((0, -1.0, 0), 2, (0, 1, 0)), ((0, 1.0, 0), 3, (0, -1, 0))):
        t, s = RC.scene_hit(np.zeros((0, 4)), 0.03, 0.97, (0.5, 0.5, 0.5), np.array([dvec], np.float64))
        assert s[0] == sid and np.isclose(t[0], 0.47, atol=1e-15)


def _frame(kind, W, H):
    scene = gen.make_scene(kind, 0)
    cam = gen.make_camera(W, H, 0)
    return scene, cam, RC.raycast(scene.spheres, scene.lo, scene.hi, cam.eye, cam.look, cam.up, cam.vfov_deg, W, H)


def test_hits_lie_on_their_surface_and_nothing_is_nearer():
    scene, cam, (x, n, wo, s) = _frame("many", 96, 64)
    S = len(scene.spheres)
    assert (s >= 0).all() and (s < S).any() and (s >= S).any()
    xd = x.astype(np.float64)
    for k in range(S):
        m = s == k
        c, R = scene.spheres[k, :3], scene.spheres[k, 3]
        assert np.allclose(np.linalg.norm(xd[m] - c, axis=1), R, atol=2e-7)                 # fp32 storage
        assert np.allclose(n[m], (xd[m] - c) / R, atol=1e-5)
        assert (np.sum(n[m] * wo[m], 1) > -1e-6).all()                                        # front side
    for p in range(5):
        m = s == S + p
        pos = scene.hi if RC.PLANE_SIDE[p] else scene.lo
        assert np.allclose(xd[m][:, RC.PLANE_AXIS[p]], pos, atol=1e-7)
    # brute force: march every ray in small steps from the eye; the first sample inside a sphere or outside the box must
    # not come before the reported hit
    o = np.asarray(cam.eye)
    t_hit = np.linalg.norm(xd - o, axis=1)
    d = -wo.astype(np.float64)
    ts = np.linspace(0.0, 1.0, 400)[None, :, None]
    pts = o + d[:, None, :] * (ts * (t_hit[:, None, None] - 2e-3))                            # strictly before the hit
    inside_box = ((pts[..., :2] > scene.lo) & (pts[..., :2] < scene.hi)).all(-1) & (pts[..., 2] > scene.lo)
    assert inside_box.all()
    for k in range(S):
        c, R = scene.spheres[k, :3], scene.spheres[k, 3]
        assert (np.linalg.norm(pts - c, axis=-1) > R - 1e-9).all()


def test_matches_the_generators_c_ray_caster():
    """Two independent implementations of the same definition (numpy here, C in gen/oo_gen.c): identical surface ids and
    identical fp32 outputs (tan() may differ in the last place between the two maths libraries: allow one fp32 ulp on a
    vanishing fraction)."""
    for kind, W, H in (("three", 160, 120), ("many", 128, 96)):
        scene, cam, (x, n, wo, s) = _frame(kind, W, H)
        q, surf = gen.raycast(scene, cam, with_surf=True)
        assert np.array_equal(s, surf)
        for a, b in ((x, q.x), (n, q.nrm), (wo, q.wo)):
            same = a == b
            assert same.mean() > 0.9999
            assert np.allclose(a, b, rtol=2e-7, atol=1e-9)
