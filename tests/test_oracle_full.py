"""Pins for oracle/oo_oracle_full.py (the NEXT rows f1-f4 of SURVEY.md §8(f)): each piece is checked against something
other than itself — closed forms, a library routine, an independent geometric construction, brute force."""
import numpy as np
import pytest

import gen
from oracle import oo_oracle as O
from oracle import oo_oracle_full as FO

torch = pytest.importorskip("torch")


def _unit(n, seed):
    r = np.random.default_rng(seed)
    v = r.normal(size=(n, 3))
    return (v / np.linalg.norm(v, axis=1, keepdims=True)).astype(np.float32)


# ------------------------------------------------------------------------------------------------ default mode


def test_default_mode_is_the_hot_path_oracle():
    w = gen.config0()
    q = w.queries
    f0, s0, _ = O.encode(w.tree, w.atlas.levels, q.x, q.wo)
    f1, dbg = FO.encode_full(w.tree, w.atlas.levels, q.x, q.nrm, q.wo, FO.Mode(), return_debug=True)
    assert np.array_equal(dbg[:, :, 0], s0)
    assert np.abs(f0 - f1).max() == 0.0
    r0 = O.query(w.tree, w.atlas.levels, w.mlp.weights, q.x, q.nrm, q.wo)
    r1 = FO.query_full(w.tree, w.atlas.levels, w.mlp.weights, q.x, q.nrm, q.wo)
    assert np.array_equal(r0, r1)


# ------------------------------------------------------------------------------------------------ f1: Eq. 10


def test_trilinear_weights_closed_form():
    x = np.array([[0.3, 0.3, 0.3], [0.0, 0.5, 1.0], [0.124, 0.876, 0.5]], np.float32)
    k, w = FO.neighbours(x, 2)
    assert np.allclose(w.sum(1), 1.0, atol=1e-15) and (w >= 0).all()
    # x = 0.3 at depth 2: p = 1.2 - 0.5 = 0.7 -> base cell 0, t = 0.7 on every axis (fp32 0.3 is 0.30000001)
    assert (k[0, 0] == [0, 0, 0]).all() and (k[0, 7] == [1, 1, 1]).all()
    assert abs(w[0, 0] - 0.3 ** 3) < 1e-6 and abs(w[0, 7] - 0.7 ** 3) < 1e-6 and abs(w[0, 1] - 0.7 * 0.09) < 1e-6
    # neighbour order j = a | b<<1 | c<<2 with a on the x axis
    assert (k[0, 1] == [1, 0, 0]).all() and (k[0, 2] == [0, 1, 0]).all() and (k[0, 4] == [0, 0, 1]).all()
    # x = 0 -> p = -1/2 -> base -1, t = 1/2 ;  x = 1 -> p = 3.5 -> base 3, t = 1/2 (neighbour 4 is outside the grid)
    assert k[1, 0, 0] == -1 and k[1, 0, 1] == 1 and k[1, 0, 2] == 3 and np.all(w[1] == 0.125)
    # a cell centre has all the weight on one neighbour
    k, w = FO.neighbours(np.array([[0.375, 0.625, 0.125]], np.float32), 2)
    assert (k[0, 0] == [1, 2, 0]).all() and w[0, 0] == 1.0


def _constant_maps(tree, values_per_level, R=2, F=1):
    """One constant map per node: level l, slot s holds values_per_level[l][s] everywhere."""
    return [np.broadcast_to(np.asarray(v, np.float64)[:, None, None, None], (len(v), R, R, F)).copy() for v in values_per_level]


def test_blend_reproduces_linear_fields_on_a_uniform_tree():
    tree = gen.build_tree(None, 3, uniform=True).set_levels([2, 3], [2, 2])
    vals = []
    for d in tree.level_depth:
        a, b = int(tree.depth_first[d]), int(tree.depth_first[d + 1])
        c = (tree.coords[a:b].astype(np.float64) + 0.5) / (1 << d)                 # cell centres
        vals.append(0.25 + 1.5 * c[:, 0] - 0.75 * c[:, 1] + 2.0 * c[:, 2])
    atlas = _constant_maps(tree, vals)
    r = np.random.default_rng(1)
    x = r.uniform(0.13, 0.87, size=(500, 3)).astype(np.float32)                    # interior: all 8 neighbours exist
    f = FO.encode_full(tree, atlas, x, _unit(500, 2), _unit(500, 3), FO.Mode(spatial="trilinear8"))
    xd = x.astype(np.float64)
    want = 0.25 + 1.5 * xd[:, 0] - 0.75 * xd[:, 1] + 2.0 * xd[:, 2]
    assert np.abs(f[:, 0] - want).max() < 1e-12 and np.abs(f[:, 1] - want).max() < 1e-12


def test_blend_equals_renormalised_grid_sample_on_sparse_trees():
    """Library special case: on per-node-constant maps Eq. 10 is  trilinear(values * mask) / trilinear(mask)  with
    zero padding, which torch.nn.functional.grid_sample (3-D, align_corners=False) computes."""
    scene = gen.make_scene("three", 0)
    tree = gen.build_tree(scene, 4).set_levels([2, 4], [2, 2])
    r = np.random.default_rng(5)
    vals = [r.uniform(-1, 1, size=s) for s in tree.level_slots]
    atlas = _constant_maps(tree, vals)
    x = r.uniform(0, 1, size=(4000, 3)).astype(np.float32)
    f, dbg = FO.encode_full(tree, atlas, x, _unit(4000, 2), _unit(4000, 3), FO.Mode(spatial="trilinear8"), return_debug=True)
    grid = torch.from_numpy(2.0 * x.astype(np.float64) - 1.0)[None, :, None, None, :]
    seen_empty = False
    for l, d in enumerate(tree.level_depth):
        n = 1 << d
        a, b = int(tree.depth_first[d]), int(tree.depth_first[d + 1])
        c = tree.coords[a:b].astype(np.int64)
        dense = np.zeros((2, n, n, n))                                            # [channel][z][y][x]
        dense[0, c[:, 2], c[:, 1], c[:, 0]] = vals[l]
        dense[1, c[:, 2], c[:, 1], c[:, 0]] = 1.0
        s = torch.nn.functional.grid_sample(torch.from_numpy(dense)[None], grid, mode="bilinear", padding_mode="zeros",
                                            align_corners=False)[0, :, :, 0, 0].numpy()
        want = np.where(s[1] > 0, s[0] / np.where(s[1] > 0, s[1], 1.0), 0.0)
        assert np.abs(f[:, l] - want).max() < 1e-12
        seen_empty |= bool((dbg[:, l] < 0).any())
        assert ((dbg[:, l] >= 0).sum(1) > 0).any()
    assert seen_empty                                                              # the test does exercise the indicator


def test_neighbour_nodes_by_linear_scan():
    scene = gen.make_scene("three", 0)
    tree = gen.build_tree(scene, 4).set_levels([3, 4], [2, 2])
    x = np.random.default_rng(7).uniform(0, 1, size=(300, 3)).astype(np.float32)
    atlas = _constant_maps(tree, [np.zeros(s) for s in tree.level_slots])
    _, dbg = FO.encode_full(tree, atlas, x, _unit(300, 2), _unit(300, 3), FO.Mode(spatial="trilinear8"), return_debug=True)
    for l, d in enumerate(tree.level_depth):
        k, _ = FO.neighbours(x, d)
        a, b = int(tree.depth_first[d]), int(tree.depth_first[d + 1])
        table = {tuple(c): s for s, c in enumerate(tree.coords[a:b].tolist())}     # brute force: every node of the level
        for i in range(x.shape[0]):
            for j in range(8):
                assert dbg[i, l, j] == table.get(tuple(k[i, j].tolist()), -1)


def test_blend_is_continuous_across_cell_faces_and_zero_when_all_empty():
    tree = gen.build_tree(None, 2, uniform=True).set_levels([1, 2], [4, 4])
    atlas = gen.make_atlas(tree, 4, "f32", 3).levels
    n = 200
    wo, nr = _unit(n, 1), _unit(n, 2)
    r = np.random.default_rng(3)
    x = r.uniform(0.05, 0.95, size=(n, 3)).astype(np.float32)
    x[:, 0] = 0.5                                                                  # a face of both levels
    eps = np.float32(2e-6)
    xa, xb = x.copy(), x.copy()
    xa[:, 0] -= eps
    xb[:, 0] += eps
    m = FO.Mode(spatial="trilinear8")
    fa = FO.encode_full(tree, atlas, xa, nr, wo, m)
    fb = FO.encode_full(tree, atlas, xb, nr, wo, m)
    assert np.abs(fa - fb).max() < 1e-4
    fn_a = FO.encode_full(tree, atlas, xa, nr, wo, FO.Mode())
    fn_b = FO.encode_full(tree, atlas, xb, nr, wo, FO.Mode())
    assert np.abs(fn_a - fn_b).max() > 0.1                                         # negative control: nearest cell jumps
    # a tree whose only branch is far from x: every neighbour absent -> zeros
    child = np.full((3, 8), -1, np.int32)
    child[0, 7] = 1
    child[1, 7] = 2
    t = gen.Tree(2, child, np.array([0, 1, 2], np.uint8), np.array([[0, 0, 0], [1, 1, 1], [3, 3, 3]], np.uint32),
                 np.array([0, 1, 2, 3])).set_levels([2], [2])
    f = FO.encode_full(t, [np.ones((1, 2, 2, 1))], np.array([[0.1, 0.1, 0.1]], np.float32), nr[:1], wo[:1], m)
    assert f[0, 0] == 0.0
    f = FO.encode_full(t, [np.ones((1, 2, 2, 1))], np.array([[0.7, 0.7, 0.7]], np.float32), nr[:1], wo[:1], m)
    assert abs(f[0, 0] - 1.0) < 1e-15                                              # one surviving neighbour, renormalised to 1


# ------------------------------------------------------------------------------------------------ f2: Eq. 6


def _tied_map(n, F, seed):
    a = np.random.default_rng(seed).uniform(-1, 1, size=(1, n + 1, n + 1, F))
    return gen.tie_vertex_map_borders(a)


def test_vertex_map_hand_examples():
    """tests/golden/vertex_taps.txt: worked by hand from Eq. 4-6 (n = 2 and n = 4)."""
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "vertex_taps.txt")) if l.strip() and not l.startswith("#")]
    for r in rows:
        n = int(r[0])
        w = np.array([[float(v) for v in r[1:4]]], np.float32)
        taps = [(int(r[4 + 3 * k]), int(r[5 + 3 * k]), float(r[6 + 3 * k])) for k in range(3)]
        ci, cj, up = FO.vertex_cell_f32(w, n)
        u = O.octa_encode(w.astype(np.float64))
        g = (u + 1) / 2 * n
        iv, jv, wg = FO.vertex_taps(ci, cj, up, g[:, 0] - ci, g[:, 1] - cj, n)
        got = sorted((int(iv[0, k]), int(jv[0, k]), round(float(wg[0, k]), 6)) for k in range(3))
        assert got == sorted((a, b, round(c, 6)) for a, b, c in taps), (r, got)


def test_vertex_map_reproduces_affine_fields_and_vertex_values():
    n, N = 8, 2000
    w = _unit(N, 11)
    jj, ii = np.meshgrid(np.arange(n + 1), np.arange(n + 1), indexing="ij")
    T = (0.5 + 0.25 * ii - 0.125 * jj)[None, :, :, None]
    h, _, _, _ = FO.dir_interp_vertex(T, np.zeros(N, np.int64), w, n)
    g = (O.octa_encode(w.astype(np.float64)) + 1) / 2 * n
    assert np.abs(h[:, 0] - (0.5 + 0.25 * g[:, 0] - 0.125 * g[:, 1])).max() < 1e-12
    # directions that land on vertices return that vertex's value
    T = _tied_map(4, 3, 0)
    for iv in range(5):
        for jv in range(5):
            d = O.octa_decode(np.array([[2.0 * iv / 4 - 1, 2.0 * jv / 4 - 1]]))
            h, _, _, _ = FO.dir_interp_vertex(T, np.zeros(1, np.int64), d.astype(np.float32), 4)
            assert np.abs(h[0] - T[0, jv, iv]).max() < 1e-6


def _octahedron_pl_interp(T, w, n):
    """Independent construction: piecewise-linear interpolation on the uniformly subdivided octahedron in 3-D.
    p = w/|w|_1 lies on the face of its sign octant; (|p_x|, |p_y|, |p_z|) are its barycentric coordinates w.r.t. the face
    vertices (+-x, +-y, +-z).  With m = n/2 subdivisions per face edge the lattice point (I, J, K)/m, I+J+K = m, sits at
    sign * (I, J, K)/m; upright small triangles have I+J+K = m-1 for the floors, inverted ones m-2."""
    m = n // 2
    w = np.asarray(w, np.float64)
    p = w / np.abs(w).sum()
    sg = np.where(p >= 0, 1.0, -1.0)
    lam = np.abs(p) * m
    fl = np.floor(lam + 1e-12).astype(int)
    fl = np.minimum(fl, m)
    fr = lam - fl
    if fl.sum() == m:                      # exactly on a lattice point
        verts, wts = [fl], [1.0]
    elif fl.sum() == m - 1:                # upright
        verts = [fl + e for e in np.eye(3, dtype=int)]
        wts = list(fr)
    else:                                  # inverted
        assert fl.sum() == m - 2
        verts = [fl + 1 - e for e in np.eye(3, dtype=int)]
        wts = list(1.0 - fr)
    out = 0.0
    for v, wt in zip(verts, wts):
        pos = sg * v / m                                           # a point of the octahedron surface
        u = O.octa_encode(pos[None])[0]
        iv, jv = int(round((u[0] + 1) / 2 * n)), int(round((u[1] + 1) / 2 * n))
        out = out + wt * T[0, jv, iv]
    return out


@pytest.mark.parametrize("n", [2, 4, 8])
def test_vertex_map_equals_piecewise_linear_interpolant_on_the_octahedron(n):
    T = _tied_map(n, 2, n)
    w = _unit(400, 20 + n)
    h, _, _, _ = FO.dir_interp_vertex(T, np.zeros(400, np.int64), w, n)
    for k in range(400):
        assert np.abs(h[k] - _octahedron_pl_interp(T, w[k], n)).max() < 1e-6, (k, w[k])
    # negative control: splitting every cell along the OTHER diagonal is a different function
    ci, cj, _ = FO.vertex_cell_f32(w, n)
    g = (O.octa_encode(w.astype(np.float64)) + 1) / 2 * n
    a, b = g[:, 0] - ci, g[:, 1] - cj
    same = (ci >= n // 2) == (cj >= n // 2)
    worst = 0.0
    for k in range(400):
        i, j, aa, bb = int(ci[k]), int(cj[k]), a[k], b[k]
        if same[k]:        # (wrongly) main diagonal
            taps = [(i, j, 1 - aa), (i + 1, j, aa - bb), (i + 1, j + 1, bb)] if aa >= bb else [(i, j, 1 - bb), (i, j + 1, bb - aa), (i + 1, j + 1, aa)]
        else:              # (wrongly) anti-diagonal
            taps = [(i, j, 1 - aa - bb), (i + 1, j, aa), (i, j + 1, bb)] if aa + bb < 1 else [(i + 1, j + 1, aa + bb - 1), (i, j + 1, 1 - aa), (i + 1, j, 1 - bb)]
        wrong = sum(wt * T[0, jv, iv] for iv, jv, wt in taps)
        worst = max(worst, float(np.abs(wrong - _octahedron_pl_interp(T, w[k], n)).max()))
    assert worst > 1e-2


def test_vertex_map_continuity_across_the_fold_needs_tied_borders():
    n = 4
    tied = _tied_map(n, 1, 3)
    untied = np.random.default_rng(3).uniform(-1, 1, size=(1, n + 1, n + 1, 1))
    r = np.random.default_rng(9)
    # pairs of directions just above / below the equator z = 0 (the boundary of the unfolded square's inner diamond is
    # interior to the map; the OUTER border is the fold through -z: pairs just either side of the planes x = 0, y = 0 with z < 0)
    t = r.uniform(0.1, 0.9, size=300)
    a = np.stack([np.full(300, 1e-6), t, -(1 - t)], 1)
    b = a.copy()
    b[:, 0] = -1e-6
    for T, bound, should_hold in ((tied, 1e-4, True), (untied, 1e-2, False)):
        ha, _, _, _ = FO.dir_interp_vertex(T, np.zeros(300, np.int64), a.astype(np.float32), n)
        hb, _, _, _ = FO.dir_interp_vertex(T, np.zeros(300, np.int64), b.astype(np.float32), n)
        gap = np.abs(ha - hb).max()
        assert (gap < bound) == should_hold, gap


# ------------------------------------------------------------------------------------------------ f3: directions


def test_mirror_direction():
    th = np.linspace(0.05, 1.5, 20)
    n = np.tile(np.array([[0, 0, 1]], np.float32), (20, 1))
    wo = np.stack([np.sin(th), 0 * th, np.cos(th)], 1).astype(np.float32)
    wr = FO.mirror_f32(n, wo)
    assert np.abs(wr - np.stack([-np.sin(th), 0 * th, np.cos(th)], 1)).max() < 1e-6
    nr, w = _unit(1000, 1), _unit(1000, 2)
    wr32, wr64 = FO.mirror_f32(nr, w).astype(np.float64), FO.mirror_f64(nr, w)
    assert np.abs(wr32 - wr64).max() < 5e-7
    assert np.abs(np.sum(wr64 * nr, 1) - np.sum(w.astype(np.float64) * nr, 1)).max() < 1e-6       # same angle to the normal (n is unit to fp32 rounding)
    assert np.abs(np.linalg.norm(wr64, axis=1) - np.linalg.norm(w.astype(np.float64), axis=1)).max() < 1e-6
    assert np.abs(FO.mirror_f32(nr, nr) - nr).max() < 1e-6                                          # wo = n is its own mirror


def test_shifted_direction_matches_eq8_eq9_and_its_limits():
    N = 500
    r = np.random.default_rng(4)
    x = r.uniform(0, 1, size=(N, 3)).astype(np.float32)
    c = ((np.floor(x * 4) + 0.5) / 4).astype(np.float32)
    wr = _unit(N, 5)
    d = r.uniform(0.25, 4.0, size=N).astype(np.float32)
    s32 = FO.shifted_f32(x, c, d, wr).astype(np.float64)
    s32 /= np.linalg.norm(s32, axis=1, keepdims=True)
    s64 = FO.shifted_f64(x, c, d, wr)                       # through the virtual point y of Eq. 8
    assert np.abs(s32 - s64).max() < 1e-5
    assert np.array_equal(FO.shifted_f32(x, c, np.zeros(N, np.float32), wr), wr)                    # d^ -> 0: the mirror direction
    far = FO.shifted_f32(x, c, np.full(N, 1e6, np.float32), wr).astype(np.float64)
    far /= np.linalg.norm(far, axis=1, keepdims=True)
    toward = (x - c).astype(np.float64)
    toward /= np.linalg.norm(toward, axis=1, keepdims=True)
    assert np.abs(far - toward).max() < 1e-4                                                       # d^ -> inf: from the cell centre to x


def test_full_mode_against_a_per_query_python_loop():
    """Composition: Eq. 9 + Eq. 6 + Eq. 10 written once more as a scalar loop over queries, neighbours and taps."""
    scene = gen.make_scene("three", 0)
    tree = gen.build_tree(scene, 4).set_levels([2, 4], [4, 2])
    atlas = gen.make_vertex_atlas(tree, 4, "f32", 0).levels
    N = 60
    r = np.random.default_rng(8)
    x = r.uniform(0, 1, size=(N, 3)).astype(np.float32)
    nr, wo = _unit(N, 1), _unit(N, 2)
    d = gen.disparity(N, 0)
    mode = FO.Mode(spatial="trilinear8", dirmap="vertex", lookup="shifted")
    f = FO.encode_full(tree, atlas, x, nr, wo, mode, disparity=d)
    F = 4
    for i in range(N):
        wr = FO.mirror_f32(nr[i], wo[i])
        for l, (dep, n) in enumerate(zip(tree.level_depth, tree.level_res)):
            nc = 1 << dep
            a0, b0 = int(tree.depth_first[dep]), int(tree.depth_first[dep + 1])
            table = {tuple(c): s for s, c in enumerate(tree.coords[a0:b0].tolist())}
            p = np.clip(x[i].astype(np.float64), 0, 1) * nc - 0.5
            k0 = np.floor(p).astype(int)
            t = p - k0
            num, den = np.zeros(F), 0.0
            for j in range(8):
                o = np.array([j & 1, (j >> 1) & 1, (j >> 2) & 1])
                kk = k0 + o
                s = table.get(tuple(kk.tolist()), -1)
                if s < 0:
                    continue
                wsp = float(np.prod(np.where(o == 1, t, 1 - t)))
                cen = ((kk + 0.5) / nc).astype(np.float32)
                wt = FO.shifted_f32(x[i], cen, d[i], wr)
                h, _, _, _ = FO.dir_interp_vertex(atlas[l], np.array([s]), wt[None], n)
                num += wsp * h[0]
                den += wsp
            want = num / den if den > 0 else np.zeros(F)
            assert np.abs(f[i, l * F:(l + 1) * F] - want).max() < 1e-12


def test_paper_attribute_vector_routing():
    """Eq. 12: g = [x, w_r, n, a, alpha] follows the L*F features; one-hot first-layer rows expose every slot."""
    w = gen.config0(n=16)
    q = w.queries
    ex = gen.albedo_roughness(16, 0)
    mode = FO.Mode(attrs="paper")
    f = FO.encode_full(w.tree, w.atlas.levels, q.x, q.nrm, q.wo, mode)
    inp = FO.mlp_input_full(f, q.x, q.nrm, q.wo, ex, mode)
    assert inp.shape[1] == 8 + 13
    wr = FO.mirror_f32(q.nrm, q.wo)
    assert np.array_equal(inp[:, 8:11], q.x.astype(np.float64)) and np.array_equal(inp[:, 11:14], wr.astype(np.float64))
    assert np.array_equal(inp[:, 14:17], q.nrm.astype(np.float64)) and np.array_equal(inp[:, 17:21], ex.astype(np.float64))
