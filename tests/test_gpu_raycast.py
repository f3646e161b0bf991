"""GPU parity of oo_raycast against oracle/oo_raycast.py: surface ids bit-exact, the fp32 queries
bit-exact (both sides follow the same double-precision operation sequence; only tan() of the field of view comes from
two maths libraries, so one fp32 ulp is allowed on a vanishing fraction), and the frame fed straight into oo_query."""
import numpy as np
import pytest

import gen
from oracle import oo_oracle as O
from oracle import oo_raycast as RC
from parity import check_rgb

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def P():
    import paper_2606_08469_b200 as P
    return P


def _compare(got, ref):
    x, n, wo, s = (t.cpu().numpy() for t in got)
    rx, rn, rwo, rs = ref
    assert np.array_equal(s.astype(np.int64), rs), "surface ids differ"
    for a, b in ((x, rx), (n, rn), (wo, rwo)):
        assert (a == b).mean() > 0.9999
        assert np.allclose(a, b, rtol=2e-7, atol=1e-9)
    return float(np.mean([(a == b).mean() for a, b in ((x, rx), (n, rn), (wo, rwo))]))


@pytest.mark.parametrize("kind,W,H", [("three", 257, 131), ("many", 192, 160), ("three", 1, 1)])
def test_raycast_matches_the_oracle(P, kind, W, H):
    scene = gen.make_scene(kind, 0)
    cam = gen.make_camera(W, H, 0)
    ctx = P.OctaOctree(0)
    ctx.oo_upload_scene(scene.spheres, scene.lo, scene.hi)
    got = ctx.oo_raycast(cam.eye, cam.look, cam.up, cam.vfov_deg, W, H, want_surf=True)
    torch.cuda.synchronize()
    ref = RC.raycast(scene.spheres, scene.lo, scene.hi, cam.eye, cam.look, cam.up, cam.vfov_deg, W, H)
    _compare(got, ref)
    ctx.close()


def test_misses_inside_spheres_and_empty_scenes(P):
    ctx = P.OctaOctree(0)
    # looking out of the open side: every ray misses; eye inside a sphere: the far root
    for spheres, eye, look in ((np.zeros((0, 4)), (0.5, 0.5, 0.5), (0.5, 0.5, 2.0)),
                               (np.array([[0.5, 0.5, 0.8, 0.3]]), (0.5, 0.5, 0.8), (0.5, 0.4, 0.2)),
                               (np.zeros((0, 4)), (0.5, 0.5, 0.9), (0.2, 0.4, 0.1))):
        ctx.oo_upload_scene(spheres, 0.03, 0.97)
        got = ctx.oo_raycast(eye, look, (0, 1, 0), 70.0, 64, 48, want_surf=True)
        torch.cuda.synchronize()
        ref = RC.raycast(spheres, 0.03, 0.97, eye, look, (0, 1, 0), 70.0, 64, 48)
        _compare(got, ref)
    assert (ref[3] >= 0).all()
    with pytest.raises(P.OOError):
        ctx.oo_raycast((0.5, 0.5, 0.5), (0.5, 0.5, 0.5), (0, 1, 0), 60.0, 4, 4)       # look == eye
    ctx.close()


def test_frame_goes_from_the_camera_to_rgb_on_the_device(P):
    """oo_raycast -> oo_query with no host copy of the queries: same RGB as the oracle evaluated on the oracle's frame."""
    w = gen.scene_workload(1, width=160, height=120, max_depth=6)
    cam = w.camera
    ctx = P.OctaOctree(0).upload_workload(w)
    ctx.oo_upload_scene(w.scene.spheres, w.scene.lo, w.scene.hi)
    x, n, wo = ctx.oo_raycast(cam.eye, cam.look, cam.up, cam.vfov_deg, cam.width, cam.height)
    rgb = ctx.oo_query(x, n, wo)
    torch.cuda.synchronize()
    rx, rn, rwo, _ = RC.raycast(w.scene.spheres, w.scene.lo, w.scene.hi, cam.eye, cam.look, cam.up, cam.vfov_deg, cam.width, cam.height)
    ref = O.query(w.tree, w.atlas.levels, w.mlp.weights, rx, rn, rwo, None, w.mlp.out_act)
    # a query whose fp32 position differs by an ulp may sit in another cell: compare where the frames agree exactly
    same = (x.cpu().numpy() == rx).all(1) & (wo.cpu().numpy() == rwo).all(1) & (n.cpu().numpy() == rn).all(1)
    assert same.mean() > 0.999
    check_rgb(rgb.cpu().numpy()[same], ref[same])
    ctx.close()


def test_full_size_frames_sampled(P):
    """The frames bench.py times (1024x1024 on the three-sphere scene, 2048x2048 on the 64-sphere scene): whole frame on
    the GPU, the oracle on every 16th scanline."""
    for kind, W, H in (("three", 1024, 1024), ("many", 2048, 2048)):
        scene = gen.make_scene(kind, 0)
        cam = gen.make_camera(W, H, 0)
        ctx = P.OctaOctree(0)
        ctx.oo_upload_scene(scene.spheres, scene.lo, scene.hi)
        got = ctx.oo_raycast(cam.eye, cam.look, cam.up, cam.vfov_deg, W, H, want_surf=True)
        torch.cuda.synchronize()
        rows = np.arange(0, H, 16)
        idx = (rows[:, None] * W + np.arange(W)[None, :]).ravel()
        ref = RC.raycast(scene.spheres, scene.lo, scene.hi, cam.eye, cam.look, cam.up, cam.vfov_deg, W, H, rows=rows)
        _compare(tuple(t[torch.from_numpy(idx).cuda()] for t in got), ref)
        ctx.close()
