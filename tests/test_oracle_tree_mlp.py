"""Pins for the oracle's quantise/descent (O1-O2), concat/MLP (O7-O8), Morton order (a1) and the end-to-end path.

Brute force (linear scan over all nodes), closed forms (uniform tree = Morton code), naive triple loops, routing
matrices, closed-form end-to-end cases (constant / per-node-constant atlases), and the two independent oracle
implementations (numpy vs C) against each other."""
import numpy as np
import pytest

import gen
from oracle import c as OC
from oracle import oo_oracle as O


def test_quantise_edges():
    D = 8
    x = np.array([[0.0, 1.0, 1.0 - 2.0 ** -24], [-0.3, 1.7, 0.5], [np.nextafter(np.float32(0.5), np.float32(0)), 0.5,
                                                                  np.nextafter(np.float32(0.5), np.float32(1))]], np.float32)
    q = O.quantise(x, D)
    assert q.tolist() == [[0, 255, 255], [0, 255, 128], [127, 128, 128]]
    # exactness: fp32 input, fp64 or fp32 arithmetic give the same cell (power-of-two scaling)
    rng = np.random.default_rng(0)
    xs = rng.uniform(0, 1, (200000, 3)).astype(np.float32)
    for D in (2, 8, 10, 16):
        q32 = np.clip(np.floor(xs * np.float32(2 ** D)), 0, 2 ** D - 1).astype(np.int64)
        assert np.array_equal(q32, O.quantise(xs, D))


def _brute_force_node(tree, q, d):
    """Linear scan: the node of depth d whose integer cell coords equal q >> (Dmax - d); -1 if none."""
    want = q >> (tree.max_depth - d)
    hit = np.nonzero((tree.depth == d) & (tree.coords == want[None, :]).all(1))[0]
    assert len(hit) <= 1
    return int(hit[0]) if len(hit) else -1


@pytest.mark.parametrize("kind", ["cfg0", "cfg0_root0", "sparse"])
def test_descent_vs_linear_scan(kind):
    if kind == "cfg0":
        tree = gen.config0().tree
    elif kind == "cfg0_root0":
        tree = gen.config0(root0_variant=True).tree
    else:
        scene = gen.make_scene("three", 3)
        tree = gen.build_tree(scene, 4).set_levels([1, 2, 4], [4, 4, 4])
        assert 100 < tree.n_nodes < 4000                        # sparse: most depth-4 cells are absent
    rng = np.random.default_rng(1)
    x = rng.uniform(0, 1, (300, 3)).astype(np.float32)
    q = O.quantise(x, tree.max_depth)
    path = O.descend(tree.child, q, tree.max_depth)
    slots = O.slots_from_path(path, tree.map_slot, tree.level_depth)
    n_absent = 0
    for k in range(len(x)):
        for d in range(tree.max_depth + 1):
            assert path[k, d] == _brute_force_node(tree, q[k], d)
        for l, d in enumerate(tree.level_depth):
            nd = _brute_force_node(tree, q[k], d)
            assert slots[k, l] == (tree.map_slot[nd] if nd >= 0 else -1)
            n_absent += nd < 0
    if kind == "sparse":
        assert n_absent > 0                                     # the absent branch (A17) is exercised
    else:
        assert n_absent == 0


def test_uniform_tree_slot_is_morton_code():
    tree = gen.build_tree(None, 3, uniform=True).set_levels([2, 3], [4, 4])
    assert tree.n_nodes == 1 + 8 + 64 + 512
    rng = np.random.default_rng(2)
    x = rng.uniform(0, 1, (2000, 3)).astype(np.float32)
    q = O.quantise(x, 3)
    slots = O.slots_from_path(O.descend(tree.child, q, 3), tree.map_slot, tree.level_depth)
    for l, d in enumerate([2, 3]):
        c = q >> (3 - d)
        code = np.zeros(len(x), np.int64)
        for b in range(d):                                      # children are created in octant order at every depth
            shift = d - 1 - b
            o = ((c[:, 0] >> shift) & 1) | (((c[:, 1] >> shift) & 1) << 1) | (((c[:, 2] >> shift) & 1) << 2)
            code = code * 8 + o
        assert np.array_equal(slots[:, l], code)


def test_octant_axis_convention():
    # o = bx | by<<1 | bz<<2: the child at +x of the root's first octant has index 1, +y index 2, +z index 4
    tree = gen.build_tree(None, 1, uniform=True).set_levels([1], [2])
    for x, o in [((0.75, 0.25, 0.25), 1), ((0.25, 0.75, 0.25), 2), ((0.25, 0.25, 0.75), 4), ((0.75, 0.75, 0.75), 7)]:
        q = O.quantise(np.array([x], np.float32), 1)
        assert O.descend(tree.child, q, 1)[0, 1] == tree.child[0, o]
        assert tuple(tree.coords[tree.child[0, o]]) == tuple(int(v > 0.5) for v in x)


def test_mlp_vs_triple_loop_and_zero_weights():
    rng = np.random.default_rng(3)
    dims = [14, 64, 64, 3]
    ws = [rng.normal(size=(dims[k + 1], dims[k])).astype(np.float16) * np.float16(0.3) for k in range(3)]
    inp = rng.normal(size=(7, 14))
    got = O.mlp(ws, inp, "exp")
    for r in range(7):
        a = list(inp[r])
        for k, W in enumerate(ws):
            b = []
            for o in range(W.shape[0]):
                acc = 0.0
                for i in range(W.shape[1]):
                    acc += float(W[o, i]) * a[i]
                b.append(max(acc, 0.0) if k < 2 else acc)
            a = b
        assert np.allclose(got[r], np.exp(a), rtol=1e-12)
    zero = [np.zeros_like(w) for w in ws]
    assert np.array_equal(O.mlp(zero, inp, "exp"), np.ones((7, 3)))
    assert np.array_equal(O.mlp(zero, inp, "none"), np.zeros((7, 3)))
    # ReLU really is applied between layers (a negative pre-activation must not propagate)
    w1 = np.array([[-1.0]], np.float16)
    assert O.mlp([w1, np.array([[1.0]], np.float16)], np.array([[2.0]]), "none")[0, 0] == 0.0


def test_concat_order_by_routing():
    """Eq. 11-13 / A7: [h_0 .. h_{L-1} | n | wo | extra]. A first layer that copies input k to hidden unit k and an
    output layer that copies hidden units exposes the position of every component."""
    L, F = 2, 4
    rng = np.random.default_rng(4)
    feats = rng.uniform(0.1, 1, (5, L * F))
    nrm, wo, ex = rng.uniform(0.1, 1, (5, 3)).astype(np.float32), rng.uniform(0.1, 1, (5, 3)).astype(np.float32), \
        rng.uniform(0.1, 1, (5, 1)).astype(np.float32)
    inp = O.mlp_input(feats, nrm, wo, ex)
    assert inp.shape == (5, L * F + 7)
    assert np.array_equal(inp[:, :8], feats) and np.array_equal(inp[:, 8:11], nrm) and np.array_equal(inp[:, 11:14], wo)
    assert np.array_equal(inp[:, 14:15], ex)
    W1 = np.zeros((64, 15), np.float16)
    for k in range(15):
        W1[k, k] = 1
    for pick in (0, 7, 8, 13, 14):
        W2 = np.zeros((3, 64), np.float16)
        W2[0, pick] = 1
        z = O.mlp([W1, W2], inp, "none")
        assert np.array_equal(z[:, 0], inp[:, pick])


def test_end_to_end_closed_forms(cfg0):
    w = cfg0
    q = w.queries
    # (1) constant atlases: h is the constant for every query, so rgb = MLP([c..c | n | wo])
    const = [np.full_like(a, 0.25 * (l + 1)) for l, a in enumerate(w.atlas.levels)]
    f, s, t = O.encode(w.tree, const, q.x, q.wo)
    assert np.array_equal(f[:, :4], np.full((q.n, 4), 0.25)) or np.abs(f[:, :4] - 0.25).max() < 1e-15
    assert np.abs(f[:, 4:] - 0.5).max() < 1e-15
    rgb = O.query(w.tree, const, w.mlp.weights, q.x, q.nrm, q.wo)
    inp = np.concatenate([np.full((q.n, 4), 0.25), np.full((q.n, 4), 0.5), q.nrm.astype(np.float64), q.wo.astype(np.float64)], 1)
    assert np.abs(rgb - O.mlp(w.mlp.weights, inp)).max() < 1e-12
    # (2) per-node-constant atlases (value = slot id): h reveals the node chosen = the cell that contains x
    ids = [np.broadcast_to(np.arange(a.shape[0], dtype=np.float32)[:, None, None, None], a.shape) for a in w.atlas.levels]
    f, s, t = O.encode(w.tree, ids, q.x, q.wo)
    cell1 = np.floor(q.x.astype(np.float64) * 2).astype(int)
    cell2 = np.floor(q.x.astype(np.float64) * 4).astype(int)
    # uniform tree built in octant order: slot at the 8-node level = octant of the root; next level = 8*parent + octant
    o1 = cell1[:, 0] | cell1[:, 1] << 1 | cell1[:, 2] << 2
    c2 = cell2 & 1
    o2 = c2[:, 0] | c2[:, 1] << 1 | c2[:, 2] << 2
    assert np.array_equal(s[:, 0], o1) and np.array_equal(s[:, 1], o1 * 8 + o2)
    assert np.abs(f[:, 0] - o1).max() < 1e-12 and np.abs(f[:, 4] - (o1 * 8 + o2)).max() < 1e-12


@pytest.mark.parametrize("name", ["cfg0", "cfg0_root0", "cfg1_small", "cfg2_small", "sparse_random"])
def test_numpy_oracle_vs_c_oracle(name, cfg0, cfg1_small):
    if name == "cfg0":
        w = cfg0
    elif name == "cfg0_root0":
        w = gen.config0(root0_variant=True)
    elif name == "cfg1_small":
        w = cfg1_small
    elif name == "cfg2_small":
        w = gen.scene_workload(2, width=160, height=90)
    else:   # random positions in a sparse tree: most fine levels are absent (A17)
        w = gen.scene_workload(1, width=64, height=64)
        w.queries = gen.random_queries(5000, 5)
    q = w.queries
    f, s, t = O.encode(w.tree, w.atlas.levels, q.x, q.wo)
    co = OC.from_workload(w)
    f2, s2, t2 = co.encode(q.x, q.wo)
    assert np.array_equal(s, s2) and np.array_equal(t, t2)
    assert np.abs(f - f2).max() < 1e-12
    rgb = O.query(w.tree, w.atlas.levels, w.mlp.weights, q.x, q.nrm, q.wo, q.extra, w.mlp.out_act)
    rgb2 = co.query(q.x, q.nrm, q.wo, q.extra)
    assert np.abs(rgb - rgb2).max() < 1e-12 * max(1.0, rgb.max())
    assert f.shape[1] == len(w.tree.level_depth) * w.atlas.F           # Eq. 11: dimension K*C
    if name == "sparse_random":
        assert (s < 0).any() and np.all(f.reshape(q.n, -1, w.atlas.F)[s < 0] == 0)
    else:
        assert (s >= 0).all()                                          # primary hits always land in existing cells
    # single-thread and multi-thread C runs agree bit for bit (queries are independent)
    assert np.array_equal(co.query(q.x, q.nrm, q.wo, q.extra, n_threads=1), rgb2)


def test_morton_keys_vs_bit_loop():
    rng = np.random.default_rng(6)
    x = rng.uniform(-0.1, 1.1, (500, 3)).astype(np.float32)
    keys = O.morton_keys(x)
    for k in range(len(x)):
        q = [min(max(int(np.floor(float(v) * 1024)), 0), 1023) for v in x[k]]
        key = 0
        for b in range(10):
            for a in range(3):
                key |= ((q[a] >> b) & 1) << (3 * b + a)
        assert key == keys[k]
    order = O.morton_order(x)
    ks = keys[order]
    assert np.all(np.diff(ks) >= 0)
    same = np.diff(ks) == 0
    assert np.all(np.diff(order)[same] > 0)                            # ties keep the original order
