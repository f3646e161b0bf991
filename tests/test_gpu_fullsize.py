"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (config 1: every query against
the C oracle; config 3: the full 10 M-node / multi-GB atlas, every one of its 4 M queries against the C oracle; config 4: every query
at 2^20, every 16th at 2^22 and 2^24; the paper's shapes: 65,536 queries of the frame against the numpy oracle of the full query)."""
import numpy as np
import pytest

import gen
from oracle import c as OC
from parity import check_features, check_indices, check_rgb

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


CHUNK = 1 << 19


def _oracle_on_every_query(co, q, rgb, slot, texel, feat):
    """RGB, slots, base texels and feature rows (host arrays, any may be None) of EVERY query of q against the C oracle, a chunk at
    a time: the oracle's fp64 feature rows of a whole 4 M-query frame would be 2.7 GB.  The RGB bars are applied per chunk (so the
    mean-abs bar holds on every 2^19 queries, not only on the whole).  Returns the worst max-abs / mean-abs RGB error."""
    worst = [0.0, 0.0]
    for lo in range(0, q.n, CHUNK):
        sl = slice(lo, min(lo + CHUNK, q.n))
        if rgb is not None:
            ref = co.query(q.x[sl], q.nrm[sl], q.wo[sl], None if q.extra is None else q.extra[sl])
            mx, mean = check_rgb(rgb[sl], ref)
            worst = [max(worst[0], mx), max(worst[1], mean)]
        if slot is not None or feat is not None:
            f, s, t = co.encode(q.x[sl], q.wo[sl])
            if slot is not None:
                check_indices(slot[sl], texel[sl], s, t)
            if feat is not None:
                check_features(feat[sl].astype(np.float32), f)
    return worst


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
    # the indices of the TIMED kernel itself (fused_tm_kernel's debug instance: same descent + gather code), all 1 M queries
    rgb_d, s_d, t_d = ctx.oo_query_debug(x, n, wo)
    assert ctx.oo_get_info()["path_last_query"] == P.PATH_FUSED_TC_TMEM and torch.equal(rgb_d, got)
    check_indices(s_d.cpu().numpy(), t_d.cpu().numpy(), s, t)
    print("cfg1 full: rgb max-abs %.3g mean-abs %.3g" % (mx, mean))


def test_config2_full_frame_all_queries():
    """configs[2] at full size: 1280x720 = 921,600 queries with the per-pixel roughness input (MLP input 39), every query
    against the C oracle; scanline order, Morton-sorted (oo_sort_queries + perm) and OO_PRESORT_BIN give the same bytes."""
    import paper_2606_08469_b200 as P
    w = gen.scene_workload(2)
    q = w.queries
    assert q.n == 1280 * 720 and q.extra is not None and q.extra.shape == (q.n, 1) and w.mlp.in_dim == 39
    co = OC.from_workload(w)
    ref = co.query(q.x, q.nrm, q.wo, q.extra)
    f, s, t = co.encode(q.x, q.wo)
    ctx = P.OctaOctree(0).upload_workload(w)
    ctx.oo_reserve(q.n)
    ctx.oo_set_presort("none")
    x, n, wo, ex = _dev(q.x), _dev(q.nrm), _dev(q.wo), _dev(q.extra)
    got, s_d, t_d = ctx.oo_query_debug(x, n, wo, ex)
    assert ctx.oo_get_info()["path_last_query"] == P.PATH_FUSED_TC_TMEM
    mx, mean = check_rgb(got.cpu().numpy(), ref)
    check_indices(s_d.cpu().numpy(), t_d.cpu().numpy(), s, t)
    plain = ctx.oo_query(x, n, wo, ex)
    assert torch.equal(plain, got)
    perm = ctx.oo_sort_queries(x)
    assert torch.equal(ctx.oo_query(x, n, wo, ex, perm=perm), plain)
    ctx.oo_set_presort("bin")
    assert torch.equal(ctx.oo_query(x, n, wo, ex), plain) and ctx.oo_get_info()["presorted_last_query"] == 1
    rgb_b, s_b, t_b = ctx.oo_query_debug(x, n, wo, ex)          # binned: index rows still land at the query's own index
    assert torch.equal(rgb_b, plain) and torch.equal(s_b, s_d) and torch.equal(t_b, t_d)
    ctx.oo_set_presort("none")
    check_features(ctx.oo_encode(x, wo).float().cpu().numpy(), f)
    print("cfg2 full: rgb max-abs %.3g mean-abs %.3g" % (mx, mean))


def test_config3_full_tree_all_queries():
    """configs[3] at full size ("cfg3: all 4 M queries for parity"): RGB of the timed kernel, the indices out of its debug
    instance, and oo_encode's feature rows and indices, EVERY one of the 4,194,304 queries against the C oracle."""
    import paper_2606_08469_b200 as P
    w = gen.scene_workload(3, width=2048, height=2048)
    assert w.tree.n_nodes > 5_000_000 and w.atlas.nbytes > 4e9
    q = w.queries
    assert q.n == 1 << 22
    ctx = P.OctaOctree(0).upload_workload(w)
    x, n, wo = _dev(q.x), _dev(q.nrm), _dev(q.wo)
    got = ctx.oo_query(x, n, wo)
    torch.cuda.synchronize()
    assert ctx.oo_get_info()["path_last_query"] == P.PATH_FUSED_TC_TMEM
    co = OC.from_workload(w)
    ctx.oo_reserve(q.n)
    rgb_d, s_d, t_d = ctx.oo_query_debug(x, n, wo)                # the timed kernel's own indices (its debug instance)
    assert torch.equal(rgb_d, got)
    fe, s_e, t_e = ctx.oo_encode(x, wo, want_debug=True)          # a different descent (descend_plan), and the feature rows
    assert torch.equal(s_d, s_e) and torch.equal(t_d, t_e)
    del rgb_d, s_e, t_e
    got = got.cpu().numpy()
    mx, mean = _oracle_on_every_query(co, q, got, s_d.cpu().numpy(), t_d.cpu().numpy(), fe.cpu().numpy())
    print("cfg3 full, all %d queries: rgb max-abs %.3g mean-abs %.3g" % (q.n, mx, mean))
    del s_d, t_d, fe
    # and a second CUDA path (features through HBM + the mma.sync MLP) within the north-star bars
    ctx.oo_set_path(P.PATH_UNFUSED)
    second = ctx.oo_query(x, n, wo).cpu().numpy()
    ctx.oo_set_path(P.PATH_AUTO)
    check_rgb(got, second.astype(np.float64))
    del second
    # incoherent distribution (config 4) on the same tree: "all queries for N <= 2^20"
    qi = gen.incoherent_queries(w.scene, 1 << 20, 0)
    xi, ni, wi = _dev(qi.x), _dev(qi.nrm), _dev(qi.wo)
    ctx.oo_set_presort("none")
    rgb_i, s_i, t_i = ctx.oo_query_debug(xi, ni, wi)
    f_i = ctx.oo_encode(xi, wi)
    ctx.oo_set_presort("bin")
    assert torch.equal(ctx.oo_query(xi, ni, wi), rgb_i) and ctx.oo_get_info()["presorted_last_query"] == 1
    mx, mean = _oracle_on_every_query(co, qi, rgb_i.cpu().numpy(), s_i.cpu().numpy(), t_i.cpu().numpy(), f_i.cpu().numpy())
    print("cfg4 2^20 incoherent, all queries: rgb max-abs %.3g mean-abs %.3g" % (mx, mean))
    del rgb_i, s_i, t_i, f_i
    # config 4 as bench.py --sweep 4 times it: 2^22 incoherent queries, unsorted and with OO_PRESORT_BIN at its default
    # threshold; the oracle on every 16th query, the two launches against each other on all of them
    qi = gen.incoherent_queries(w.scene, 1 << 22, 0)
    xi, ni, wi = _dev(qi.x), _dev(qi.nrm), _dev(qi.wo)
    ctx.oo_set_presort("none")
    plain = ctx.oo_query(xi, ni, wi)
    ctx.oo_reserve(qi.n)
    ctx.oo_set_presort("bin")
    binned = ctx.oo_query(xi, ni, wi)
    assert ctx.oo_get_info()["presorted_last_query"] == 1
    assert torch.equal(plain, binned)
    idx = np.arange(0, qi.n, 16)
    qs = qi.take(idx)
    fb = ctx.oo_encode(xi, wi)
    assert ctx.oo_get_info()["presorted_last_encode"] == 1
    ctx.oo_set_presort("none")
    assert torch.equal(fb, ctx.oo_encode(xi, wi))
    _oracle_on_every_query(co, qs, binned.cpu().numpy()[idx], None, None, None)
    f_ref = np.concatenate([co.encode(qs.x[k:k + CHUNK], qs.wo[k:k + CHUNK])[0] for k in range(0, qs.n, CHUNK)])
    check_features(fb[torch.from_numpy(idx).cuda()].float().cpu().numpy(), f_ref)


def test_paper_shapes_full_frame_sampled_queries():
    """The paper's own configuration at full size (bench.py --sweep 8: depths 2..9, ~2 M nodes, ~1 GB of fp32 vertex maps,
    all of f1-f4 on, decoder 4 x 128, 1024x1024 frame): the whole frame on the GPU, the numpy oracle on a sample of
    queries spread over the frame."""
    import paper_2606_08469_b200 as P
    from oracle import oo_oracle_full as FO
    w = gen.paper_workload()
    q, d = w.queries, w.meta["disparity"]
    assert q.n == 1024 * 1024 and w.tree.level_depth == list(range(2, 10)) and w.atlas.nbytes > 9e8
    ctx = P.OctaOctree(0)
    ctx.oo_upload_tree(w.tree, w.atlas.levels, "f32", dirmap="vertex")
    ctx.oo_upload_mlp(w.mlp.weights, w.mlp.out_act)
    ctx.oo_set_mode("trilinear8", "shifted", "paper")
    x, n, wo, ex, dd = _dev(q.x), _dev(q.nrm), _dev(q.wo), _dev(q.extra), _dev(d)
    got = ctx.oo_query(x, n, wo, ex, disparity=dd)
    feat, slots, _ = ctx.oo_encode_full(x, n, wo, dd, want_debug=True)
    torch.cuda.synchronize()
    assert ctx.oo_get_info()["path_last_query"] == P.PATH_FULL
    idx = np.arange(0, q.n, 16)                                    # 65,536 queries across the whole frame
    qs = q.take(idx)
    mode = FO.Mode("trilinear8", "vertex", "shifted", "paper")
    ref_f, ref_s = FO.encode_full(w.tree, w.atlas.levels, qs.x, qs.nrm, qs.wo, mode, d[idx], return_debug=True)
    ref = FO.query_full(w.tree, w.atlas.levels, w.mlp.weights, qs.x, qs.nrm, qs.wo, qs.extra, "exp", mode, d[idx])
    assert np.array_equal(slots.cpu().numpy()[idx].astype(np.int64), ref_s)
    # the fused kernel's own neighbour slots and index decisions (its debug instance) against oo_encode_full's, all 1 M queries
    rgb_d, s_d, c_d = ctx.oo_query_debug(x, n, wo, ex, disparity=dd)
    _, _, cells = ctx.oo_encode_full(x, n, wo, dd, want_debug=True)
    assert torch.equal(rgb_d, got) and torch.equal(s_d, slots) and torch.equal(c_d, cells)
    del rgb_d, s_d, c_d, cells
    check_features(feat.cpu().numpy()[idx], ref_f)
    mx, mean = check_rgb(got.cpu().numpy()[idx], ref)
    print("paper shapes full frame: rgb max-abs %.3g mean-abs %.3g on %d sampled queries" % (mx, mean, len(idx)))


@pytest.mark.parametrize("dist", ["coherent", "incoherent"])
def test_config4_2pow24_queries(dist):
    """configs[4] at its largest batch, 2^24 queries on the config-3 cache, as bench.py --sweep 4 times it: the coherent
    stream (screen-order hits of a 4096x4096 frame) and the incoherent one (area-weighted surface samples, random order).
    The oracle on every 16th query (1 M of them); the unsorted and the OO_PRESORT_BIN call against each other on all 16.8 M queries, bit
    for bit; the fused kernel's own indices against oo_encode's on all of them."""
    import paper_2606_08469_b200 as P
    w = gen.scene_workload(3, seed=0, width=64, height=64)
    n = 1 << 24
    q = gen.raycast(w.scene, gen.make_camera(4096, 4096, 0)) if dist == "coherent" else gen.incoherent_queries(w.scene, n, 0)
    assert q.n == n
    ctx = P.OctaOctree(0).upload_workload(w)
    ctx.oo_reserve(n)
    ctx.oo_set_presort("none")
    x, nr, wo = _dev(q.x), _dev(q.nrm), _dev(q.wo)
    plain = ctx.oo_query(x, nr, wo)
    assert ctx.oo_get_info()["path_last_query"] == P.PATH_FUSED_TC_TMEM
    ctx.oo_set_presort("bin")
    binned = ctx.oo_query(x, nr, wo)
    assert ctx.oo_get_info()["presorted_last_query"] == 1
    assert torch.equal(plain, binned)
    del binned
    ctx.oo_set_presort("none")
    idx = np.arange(0, n, 16)                                    # "a stride-16 subsample of the 2^24 batch" = 1,048,576 queries
    qs = q.take(idx)
    co = OC.from_workload(w)
    rgb_d, s_d, t_d = ctx.oo_query_debug(x, nr, wo)
    assert torch.equal(rgb_d, plain)
    del rgb_d
    fe, s_e, t_e = ctx.oo_encode(x, wo, want_debug=True)
    assert torch.equal(s_d, s_e) and torch.equal(t_d, t_e)
    del s_e, t_e
    mx, mean = _oracle_on_every_query(co, qs, plain.cpu().numpy()[idx], s_d[::16].cpu().numpy(), t_d[::16].cpu().numpy(),
                                      fe[::16].cpu().numpy())
    print("cfg4 2^24 %s: rgb max-abs %.3g mean-abs %.3g on %d sampled queries" % (dist, mx, mean, len(idx)))
