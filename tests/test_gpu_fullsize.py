"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (config 1: every query against
the C oracle; config 3: the full 10 M-node / multi-GB atlas, oracle on a sample of queries)."""
import numpy as np
import pytest

import gen
from oracle import c as OC
from parity import check_features, check_indices, check_rgb

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_config1_full_frame_all_queries():
    import paper_2606_08469_b200 as P
    w = gen.scene_workload(1)
    q = w.queries
    assert q.n == 1024 * 1024
    co = OC.from_workload(w)
    ref = co.query(q.x, q.nrm, q.wo)
    f, s, t = co.encode(q.x, q.wo)
    assert (s >= 0).all()
    ctx = P.OctaOctree(0).upload_workload(w)
    x, n, wo = _dev(q.x), _dev(q.nrm), _dev(q.wo)
    got = ctx.oo_query(x, n, wo)
    torch.cuda.synchronize()
    assert ctx.oo_get_info()["path_last_query"] == P.PATH_FUSED_TC_TMEM
    mx, mean = check_rgb(got.cpu().numpy(), ref)
    fe, sl, tx = ctx.oo_encode(x, wo, want_debug=True)
    check_indices(sl.cpu().numpy(), tx.cpu().numpy(), s, t)
    check_features(fe.float().cpu().numpy(), f)
    print("cfg1 full: rgb max-abs %.3g mean-abs %.3g" % (mx, mean))


def test_config3_full_tree_sampled_queries():
    import paper_2606_08469_b200 as P
    w = gen.scene_workload(3, width=2048, height=2048)
    assert w.tree.n_nodes > 5_000_000 and w.atlas.nbytes > 4e9
    q = w.queries
    ctx = P.OctaOctree(0).upload_workload(w)
    x, n, wo = _dev(q.x), _dev(q.nrm), _dev(q.wo)
    got = ctx.oo_query(x, n, wo)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    idx = np.arange(0, q.n, 61)                                  # ~69 k sampled queries across the whole frame
    qs = q.take(idx)
    co = OC.from_workload(w)
    ref = co.query(qs.x, qs.nrm, qs.wo)
    check_rgb(got[idx], ref)
    f, s, t = co.encode(qs.x, qs.wo)
    fe, sl, tx = ctx.oo_encode(_dev(qs.x), _dev(qs.wo), want_debug=True)
    check_indices(sl.cpu().numpy(), tx.cpu().numpy(), s, t)
    check_features(fe.float().cpu().numpy(), f)
    # incoherent distribution (config 4) on the same tree
    qi = gen.incoherent_queries(w.scene, 1 << 16, 0)
    ref = co.query(qi.x, qi.nrm, qi.wo)
    check_rgb(ctx.oo_query(_dev(qi.x), _dev(qi.nrm), _dev(qi.wo)).cpu().numpy(), ref)
