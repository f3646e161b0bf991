"""GPU parity of the disparity predictor g_psi (Eq. 7) against oracle/oo_hashgrid.py
through the C ABI (oo_upload_disparity, oo_predict_disparity), and of the full query that predicts d^ itself
(OO_LOOKUP_SHIFTED with queries.disparity == NULL).

What is compared: hash-grid features within 1e-3 (fp16 entries, fp32 accumulate: the north-star feature bound); d^ within
DISPARITY_REL relative (tests/parity.py: fp16 activations perturb z by ~1e-3 and d^ = exp(z)).  The composition is covered
link by link, because d^ feeds integer decisions downstream (the shifted direction picks texels) and the two sides' d^
differ in the last fp16 bits: (1) GPU d^ vs the oracle's d^ [here], (2) the GPU full query given a d^ vs the oracle given
the same d^ [tests/test_gpu_full.py], (3) the GPU full query predicting d^ internally is BIT-identical to the GPU full query
fed the output of oo_predict_disparity [here].  An end-to-end RGB comparison against the fully composed oracle is added on
a cache smooth enough that those last bits cannot matter beyond the RGB bound."""
import numpy as np
import pytest

import gen
from oracle import oo_hashgrid as HG
from oracle import oo_oracle_full as FO
from parity import DISPARITY_REL, FEATURE_ATOL, check_rgb

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def P():
    import paper_2606_08469_b200 as P
    return P


def _cu(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _ctx(P, net):
    ctx = P.OctaOctree(0)
    ctx.oo_upload_disparity(net.res, net.hash_log2, net.tables, net.weights)
    return ctx


def _check_net(P, net, q):
    grid = HG.HashGrid(net.res, net.hash_log2, net.tables)
    ref_e = HG.encode(grid, q.x)
    ref_d = HG.disparity(grid, net.weights, q.x, q.nrm, q.wo)
    ctx = _ctx(P, net)
    d, e = ctx.oo_predict_disparity(_cu(q.x), _cu(q.nrm), _cu(q.wo), want_features=True)
    torch.cuda.synchronize()
    e, d = e.cpu().numpy().astype(np.float64), d.cpu().numpy().astype(np.float64)
    assert np.abs(e - ref_e).max() <= FEATURE_ATOL, "hash-grid features: %.3g" % np.abs(e - ref_e).max()
    rel = np.abs(d - ref_d) / ref_d
    assert np.isfinite(d).all() and rel.max() <= DISPARITY_REL, "d^ relative error %.3g" % rel.max()
    ctx.close()
    return float(np.abs(e - ref_e).max()), float(rel.max())


def _edge_positions(q):
    x = q.x.copy()
    special = np.array([[0, 0, 0], [1, 1, 1], [0, 1, 0.5], [-0.25, 0.5, 1.5], [0.125, 0.375, 0.625], [1.0 - 2.0 ** -24, 0.5, 0.5],
                        [0.5, 0.5, 0.5], [2.0 ** -30, 0.3, 0.9], [1.0 / 3.0, 2.0 / 3.0, 0.1]], np.float32)
    x[: len(special)] = special
    return gen.Queries(x, q.nrm, q.wo, q.extra)


def test_default_predictor_random_queries(P):
    """8 levels 16..512, 2^17-entry tables (3 dense + 5 hashed levels), 2 x 64: N = 20,000 + 37 (ragged last tile) queries,
    degenerate positions included."""
    net = gen.make_disparity_net(0)
    q = _edge_positions(gen.random_queries(20037, 1))
    e_err, d_err = _check_net(P, net, q)
    print("default g_psi: feature max-abs %.3g, d^ max-rel %.3g" % (e_err, d_err))


@pytest.mark.parametrize("kw", [dict(n_levels=1, n_min=8, n_max=8), dict(n_levels=16, n_min=4, n_max=1024, hash_log2=14),
                                dict(n_levels=4, n_min=2, n_max=16, hash_log2=20), dict(n_levels=4, n_min=64, n_max=512, hash_log2=10),
                                dict(n_levels=8, n_hidden=1), dict(n_levels=6, n_hidden=3), dict(n_levels=13, n_min=16, n_max=300),
                                dict(res=[64, 4, 128, 8, 5], hash_log2=12), dict(n_levels=7, n_min=4, n_max=256, hash_log2=12)],
                         ids=["one-level", "sixteen-levels", "all-dense", "all-hashed-tiny-table", "one-hidden", "three-hidden", "k1-is-32",
                              "dense-and-hashed-interleaved", "ragged-batches"])
def test_predictor_shapes(P, kw):
    net = gen.make_disparity_net(2, **kw)
    q = _edge_positions(gen.random_queries(3000, 3))
    _check_net(P, net, q)


@pytest.mark.parametrize("n", [0, 1, 127, 128, 129, 640 * 148 + 5])
def test_predictor_sizes(P, n):
    net = gen.make_disparity_net(4, n_levels=4, n_min=8, n_max=64, hash_log2=12)
    ctx = _ctx(P, net)
    if n == 0:
        z = torch.empty((0, 3), device="cuda")
        assert ctx.oo_predict_disparity(z, z, z).numel() == 0
        return
    q = gen.random_queries(n, 5)
    _check_net(P, net, q)


def test_predictor_on_a_frame(P):
    """The config-1 recipe's primary hits (coherent positions on surfaces) at 320 x 200."""
    w = gen.scene_workload(1, width=320, height=200)
    _check_net(P, gen.make_disparity_net(0), w.queries)


def test_errors(P):
    net = gen.make_disparity_net(0, n_levels=2, n_min=4, n_max=8)
    ctx = P.OctaOctree(0)
    q = gen.random_queries(16, 0)
    with pytest.raises(P.OOError) as e:
        ctx.oo_predict_disparity(_cu(q.x), _cu(q.nrm), _cu(q.wo))
    assert e.value.status == 2                                   # OO_ERR_NOT_READY: nothing uploaded
    with pytest.raises(P.OOError) as e:
        ctx.oo_upload_disparity(net.res, 2, net.tables, net.weights)
    assert e.value.status == 1                                   # hash_log2 out of range
    with pytest.raises(P.OOError) as e:
        ctx.oo_upload_disparity([0, 8], net.hash_log2, net.tables, net.weights)
    assert e.value.status == 1
    t4 = [np.zeros((t.shape[0], 4), np.float16) for t in net.tables]
    with pytest.raises(P.OOError) as e:
        ctx.oo_upload_disparity(net.res, net.hash_log2, t4, net.weights)
    assert e.value.status == 3                                   # OO_ERR_UNSUPPORTED: 4 features per entry


def _paper_small(seed=0, res=None):
    """The paper-shape recipe reduced for the oracle: depths 2..5, vertex maps, C = 4 fp32, Eq. 12 attributes, 4 x 128."""
    return gen.paper_workload(seed=seed, width=96, height=64, depths=[2, 3, 4, 5], res=res or [32, 16, 8, 4])


def test_full_query_predicts_the_disparity_itself(P):
    """Link (3): OO_LOOKUP_SHIFTED with queries.disparity == NULL == the same query fed oo_predict_disparity's output, bit
    for bit, through oo_query, oo_encode_full and oo_query_host; without a predictor the call is refused."""
    w = _paper_small()
    q = w.queries
    net = gen.make_disparity_net(0)
    ctx = P.OctaOctree(0)
    ctx.oo_upload_tree(w.tree, w.atlas.levels, w.atlas.dtype, dirmap="vertex")
    ctx.oo_upload_mlp(w.mlp.weights, w.mlp.out_act)
    ctx.oo_set_mode("trilinear8", "shifted", "paper")
    x, n, wo, ex = _cu(q.x), _cu(q.nrm), _cu(q.wo), _cu(q.extra)
    with pytest.raises(P.OOError) as e:
        ctx.oo_query(x, n, wo, ex)
    assert e.value.status == 1
    ctx.oo_upload_disparity(net.res, net.hash_log2, net.tables, net.weights)
    with pytest.raises(P.OOError) as e:
        ctx.oo_query(x, n, wo, ex)
    assert e.value.status == 2                                   # scratch for d^: oo_reserve first
    ctx.oo_reserve(q.n)
    d = ctx.oo_predict_disparity(x, n, wo)
    l0 = ctx.oo_get_info()["query_launches"]
    own = ctx.oo_query(x, n, wo, ex)
    assert ctx.oo_get_info()["query_launches"] - l0 == 2         # predictor + fused full query
    fed = ctx.oo_query(x, n, wo, ex, disparity=d)
    assert torch.equal(own, fed)
    f_own, s_own, c_own = ctx.oo_encode_full(x, n, wo, None, want_debug=True)
    f_fed, s_fed, c_fed = ctx.oo_encode_full(x, n, wo, d, want_debug=True)
    assert torch.equal(f_own, f_fed) and torch.equal(s_own, s_fed) and torch.equal(c_own, c_fed)
    host = ctx.oo_query_host(q.x, q.nrm, q.wo, q.extra)
    assert np.array_equal(host.numpy(), own.cpu().numpy())
    ctx.close()


def test_end_to_end_against_the_composed_oracle_on_a_smooth_cache(P):
    """oracle g_psi -> oracle full query  vs  GPU g_psi -> GPU full query, on coarse angular maps (R = 4, 4, 2, 2 intervals:
    the interpolant moves by < 0.1 per unit of octahedral coordinate, and a 5e-3 relative change of d^ moves the shifted
    direction by < 1e-2), so that the last bits of d^ stay inside the RGB bound."""
    w = _paper_small(res=[4, 4, 2, 2])
    q = w.queries
    net = gen.make_disparity_net(0)
    mode = FO.Mode("trilinear8", "vertex", "shifted", "paper")
    d_ref = HG.disparity(HG.HashGrid(net.res, net.hash_log2, net.tables), net.weights, q.x, q.nrm, q.wo).astype(np.float32)
    ref = FO.query_full(w.tree, w.atlas.levels, w.mlp.weights, q.x, q.nrm, q.wo, q.extra, w.mlp.out_act, mode, d_ref)
    ctx = P.OctaOctree(0)
    ctx.oo_upload_tree(w.tree, w.atlas.levels, w.atlas.dtype, dirmap="vertex")
    ctx.oo_upload_mlp(w.mlp.weights, w.mlp.out_act)
    ctx.oo_upload_disparity(net.res, net.hash_log2, net.tables, net.weights)
    ctx.oo_set_mode("trilinear8", "shifted", "paper")
    ctx.oo_reserve(q.n)
    rgb = ctx.oo_query(_cu(q.x), _cu(q.nrm), _cu(q.wo), _cu(q.extra))
    torch.cuda.synchronize()
    err = check_rgb(rgb.cpu().numpy(), ref)
    print("composed g_psi + full query: rgb max-abs %.3g mean-abs %.3g" % err)
    ctx.close()
