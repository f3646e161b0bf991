"""include/oo.h promises for inputs it does not check per query — non-finite values, wo = 0, denormals, values whose sums overflow —
"result undefined, never a crash".  These tests feed such queries, scattered among valid ones, through every kernel path, the binned
order, the host entry point in both of its modes, the full query and the disparity predictor, and assert what the promise means:
every call returns OO_OK, the device is healthy afterwards (no sticky CUDA error: the next call works), the rows of the VALID queries
are bit-identical to a run that never saw the bad ones (queries are independent), and nothing is written past the end of an output.
Also here: repeated calls on one context give the same bytes (the stand-in for a race detector), and two
contexts on two streams — the header's stated way to overlap work — give the serial results."""
import numpy as np
import pytest

import gen

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

GUARD = 64
BAD = [np.nan, np.inf, -np.inf, 0.0, 1e-42, 1e38, -1e38, 3e38]      # 1e-42: denormal; 3e38: |a|+|b| overflows


@pytest.fixture(scope="module")
def P():
    import paper_2606_08469_b200 as P
    return P


def _cu(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _poison(q, disparity=None, stride=37):
    """A copy of the queries in which every stride-th one carries a bad value in one of its fields: the field, the value and
    whether one or all components get it cycle independently, so every combination occurs.  Returns (queries, disparity, valid mask)."""
    x, nrm, wo = q.x.copy(), q.nrm.copy(), q.wo.copy()
    extra = None if q.extra is None else q.extra.copy()
    d = None if disparity is None else disparity.copy()
    fields = [x, nrm, wo] + ([extra] if extra is not None else []) + ([d] if d is not None else [])
    bad = np.arange(5, q.n, stride)
    for k, i in enumerate(bad):
        a = fields[k % len(fields)]
        v = BAD[(k // len(fields)) % len(BAD)]
        if a.ndim == 1:
            a[i] = v
        elif (k // (len(fields) * len(BAD))) % 2 == 0:
            a[i, :] = v
        else:
            a[i, k % a.shape[1]] = v
    valid = np.ones(q.n, bool)
    valid[bad] = False
    return gen.Queries(x, nrm, wo, extra), d, valid


def _guarded(n, c, dtype=torch.float32):
    buf = torch.full((n + GUARD, c), -123.0, dtype=dtype, device="cuda")
    return buf, buf[:n]


def _same_valid_rows(got, clean, valid, what):
    got, clean = got.cpu().numpy(), clean.cpu().numpy()
    assert np.array_equal(got[valid], clean[valid]), "%s: a valid query's row changed because of its neighbours' bad inputs" % what


def test_bad_inputs_on_every_hot_path(P):
    w = gen.scene_workload(2, width=160, height=90)                    # 14,400 queries with the roughness extra
    q = w.queries
    qb, _, valid = _poison(q)
    assert (~valid).sum() > 300
    ctx = P.OctaOctree(0).upload_workload(w)
    ctx.oo_reserve(q.n)
    dev = lambda qq: (_cu(qq.x), _cu(qq.nrm), _cu(qq.wo), _cu(qq.extra))
    xc, nc, wc, ec = dev(q)
    xb, nb, wb, eb = dev(qb)
    paths = [P.PATH_GENERIC, P.PATH_UNFUSED, P.PATH_FUSED_MMA, P.PATH_FUSED_TC, P.PATH_FUSED_TC_TMEM]
    for path in paths:
        for presort in ("none", "bin"):
            ctx.oo_set_path(path)
            ctx.oo_set_presort(presort, min_queries=1)
            try:
                clean = ctx.oo_query(xc, nc, wc, ec)
            except P.OOError as e:
                assert e.status == 3                                   # no instance of that kernel for this shape
                continue
            buf, rgb = _guarded(q.n, 3)
            ctx.oo_query(xb, nb, wb, eb, rgb=rgb)                      # raises unless OO_OK
            torch.cuda.synchronize()                                   # raises on a sticky error
            assert ctx.oo_get_info()["presorted_last_query"] == (1 if presort == "bin" else 0)
            _same_valid_rows(rgb, clean, valid, "oo_query path %d presort %s" % (path, presort))
            assert bool((buf[q.n:] == -123.0).all())
            assert torch.equal(ctx.oo_query(xc, nc, wc, ec), clean)    # the context is as good as before
            rgb_d, s_d, t_d = ctx.oo_query_debug(xb, nb, wb, eb)       # the debug instances take the same inputs
            torch.cuda.synchronize()
            _same_valid_rows(rgb_d, clean, valid, "oo_query_debug path %d" % path)
            R = torch.tensor(w.tree.level_res, device="cuda").view(1, -1, 1)
            assert bool((t_d >= -1).all()) and bool((t_d.int() < R).all()), "a bad direction left the map"
    # oo_encode: both specialised kernels and the generic one
    for path, presort in ((P.PATH_GENERIC, "none"), (P.PATH_UNFUSED, "none"), (P.PATH_UNFUSED, "bin")):
        ctx.oo_set_path(path)
        ctx.oo_set_presort(presort, min_queries=1)
        clean = ctx.oo_encode(xc, wc)
        buf, feat = _guarded(q.n, clean.shape[1], torch.float16)
        ctx.oo_encode(xb, wb, features=feat)
        torch.cuda.synchronize()
        _same_valid_rows(feat, clean, valid, "oo_encode path %d presort %s" % (path, presort))
        assert bool((buf[q.n:] == -123.0).all())
    # oo_query_host, zero-copy launch and copy pipeline
    ctx.oo_set_path(P.PATH_AUTO)
    ctx.oo_set_presort("none")
    clean = ctx.oo_query(xc, nc, wc, ec)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    for zero_copy in (True, False):
        ctx.oo_set_host_zero_copy(zero_copy)
        hrgb = torch.full((q.n + GUARD, 3), -123.0).pin_memory()
        ctx.oo_query_host(pin(qb.x), pin(qb.nrm), pin(qb.wo), pin(qb.extra), rgb=hrgb[:q.n])
        torch.cuda.synchronize()
        assert np.array_equal(hrgb[:q.n].numpy()[valid], clean.cpu().numpy()[valid]) and bool((hrgb[q.n:] == -123.0).all())
    ctx.oo_set_host_zero_copy(True)
    assert torch.equal(ctx.oo_query(xc, nc, wc, ec), clean)
    ctx.close()


def test_bad_inputs_on_the_full_query_and_the_predictor(P):
    w = gen.scene_workload(1, width=128, height=96, max_depth=6)
    q = w.queries
    q.extra = gen.albedo_roughness(q.n, 0)
    d = gen.disparity(q.n, 0)
    qb, db, valid = _poison(q, d)
    dev = lambda qq, dd: (_cu(qq.x), _cu(qq.nrm), _cu(qq.wo), _cu(qq.extra), _cu(dd))
    xc, nc, wc, ec, dc = dev(q, d)
    xb, nb, wb, eb, dbd = dev(qb, db)
    net = gen.make_disparity_net(0)
    for dirmap, width in (("vertex", 64), ("texel", 128)):
        atlas = (gen.make_vertex_atlas(w.tree, 8, "f16", 0) if dirmap == "vertex" else w.atlas).levels
        mlp = gen.make_mlp(24 + 9 + 4, 4, 0, width=width)
        ctx = P.OctaOctree(0)
        ctx.oo_upload_tree(w.tree, atlas, "f16", dirmap=dirmap)
        ctx.oo_upload_mlp(mlp.weights, mlp.out_act)
        ctx.oo_upload_disparity(net.res, net.hash_log2, net.tables, net.weights)
        ctx.oo_reserve(q.n)
        for lookup in ("shifted", "mirror"):
            for presort in ("none", "bin"):
                ctx.oo_set_mode("trilinear8", lookup, "paper")
                ctx.oo_set_presort(presort, min_queries=1)
                what = "%s maps, width %d, %s, presort %s" % (dirmap, width, lookup, presort)
                clean = ctx.oo_query(xc, nc, wc, ec, disparity=dc)
                buf, rgb = _guarded(q.n, 3)
                ctx.oo_query(xb, nb, wb, eb, rgb=rgb, disparity=dbd)
                torch.cuda.synchronize()
                assert ctx.oo_get_info()["path_last_query"] == P.PATH_FULL
                _same_valid_rows(rgb, clean, valid, "full query, " + what)
                assert bool((buf[q.n:] == -123.0).all())
                f_clean = ctx.oo_encode_full(xc, nc, wc, dc)
                f_bad = ctx.oo_encode_full(xb, nb, wb, dbd)
                torch.cuda.synchronize()
                _same_valid_rows(f_bad, f_clean, valid, "oo_encode_full, " + what)
                rgb_d = ctx.oo_query_debug(xb, nb, wb, eb, disparity=dbd)[0]
                torch.cuda.synchronize()
                _same_valid_rows(rgb_d, clean, valid, "full query debug instance, " + what)
                if lookup == "shifted":                                # d^ predicted inside the call from the (bad) positions
                    clean_p = ctx.oo_query(xc, nc, wc, ec)
                    bad_p = ctx.oo_query(xb, nb, wb, eb)
                    torch.cuda.synchronize()
                    _same_valid_rows(bad_p, clean_p, valid, "full query with predicted d^, " + what)
        d_clean = ctx.oo_predict_disparity(xc, nc, wc)
        d_bad = ctx.oo_predict_disparity(xb, nb, wb)
        torch.cuda.synchronize()
        _same_valid_rows(d_bad.view(-1, 1), d_clean.view(-1, 1), valid, "oo_predict_disparity")
        ctx.oo_set_presort("none")
        assert torch.equal(ctx.oo_query(xc, nc, wc, ec, disparity=dc), ctx.oo_query(xc, nc, wc, ec, disparity=dc))
        ctx.close()


def test_repeated_calls_are_bit_identical(P):
    """200 back-to-back calls on one context, no synchronisation in between, alternating two batches of different sizes: every result
    equals the first of its kind.  A race in the mbarrier / tensor-memory pipeline, a stale scratch row or a slot handed back too
    early shows up here as a differing byte."""
    w = gen.scene_workload(1, width=512, height=300)
    q = w.queries
    ctx = P.OctaOctree(0).upload_workload(w)
    ctx.oo_reserve(q.n)
    x, n, wo = _cu(q.x), _cu(q.nrm), _cu(q.wo)
    m = 77_777
    for presort in ("none", "bin"):
        ctx.oo_set_presort(presort, min_queries=1)
        ref_a, ref_b = ctx.oo_query(x, n, wo), ctx.oo_query(x[:m], n[:m], wo[:m])
        outs = [(ctx.oo_query(x, n, wo), ctx.oo_query(x[:m], n[:m], wo[:m])) for _ in range(100)]
        torch.cuda.synchronize()
        assert torch.equal(ref_b, ref_a[:m])
        assert all(torch.equal(a, ref_a) and torch.equal(b, ref_b) for a, b in outs), "presort %s" % presort
    ctx.close()


def test_two_contexts_on_two_streams_overlap_safely(P):
    """include/oo.h: work that is to overlap on several streams takes one context per stream.  Two contexts with different caches,
    each on its own stream, 50 interleaved calls each (binned, so both use their context-owned scratch): the serial results."""
    w1 = gen.scene_workload(1, width=400, height=300)
    w2 = gen.scene_workload(3, width=300, height=200, max_depth=8)
    ctxs, data, refs = [], [], []
    for w in (w1, w2):
        c = P.OctaOctree(0).upload_workload(w)
        c.oo_reserve(w.queries.n)
        c.oo_set_presort("bin", min_queries=1)
        t = (_cu(w.queries.x), _cu(w.queries.nrm), _cu(w.queries.wo))
        ctxs.append(c)
        data.append(t)
        refs.append(c.oo_query(*t))
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [[], []]
    for _ in range(50):
        for k in (0, 1):
            with torch.cuda.stream(streams[k]):
                outs[k].append(ctxs[k].oo_query(*data[k]))
    torch.cuda.synchronize()
    for k in (0, 1):
        assert all(torch.equal(o, refs[k]) for o in outs[k]), "context %d" % k
        ctxs[k].close()
