"""Host-side checks of the seeded input generators (gen/): determinism, storage rounding, tree invariants, and
that every primary hit of the analytic scene lands in existing cells at every used level (A17: expected 0 misses)."""
import numpy as np

import gen
from oracle import oo_oracle as O


def test_counter_based_rng_is_deterministic_and_sliceable():
    a = gen.u01(0, 1, 1000)
    assert np.array_equal(a, gen.u01(0, 1, 1000))
    assert np.array_equal(a[300:700], gen.u01(0, 1, 400, first=300))          # any element independently
    assert not np.array_equal(a, gen.u01(1, 1, 1000)) and not np.array_equal(a, gen.u01(0, 2, 1000))
    assert 0 <= a.min() and a.max() < 1
    n = gen.normal(0, 2, 400000)
    assert abs(n.mean()) < 0.01 and abs(n.std() - 1) < 0.01
    h = gen.normal_f16(0, 3, 1000, 0.1)
    assert np.array_equal(h, gen.normal_f16(0, 3, 1000, 0.1)) and h.dtype == np.float16


def test_f16_rounding_matches_numpy_rne():
    a = np.concatenate([gen.normal(0, 1, 50000) * s for s in (1e-9, 6e-8, 1e-5, 1e-3, 0.1, 1, 100, 6e4)])
    a = np.concatenate([a, [0.0, -0.0, 65504.0, 65519.9, 65520.0, 2.0 ** -24, 2.0 ** -25, 2.0 ** -25 * 1.0001, 1.00048828125]])
    with np.errstate(over="ignore"):
        ref = a.astype(np.float16)
    assert np.array_equal(gen.f64_to_f16(a).view(np.uint16), ref.view(np.uint16))


def test_tree_invariants(cfg1_small):
    t = cfg1_small.tree
    assert t.max_depth == 8 and t.level_depth == [2, 4, 6, 8] and t.level_res == [32, 16, 8, 4]
    assert 300_000 < t.n_nodes < 700_000                       # literal build rule: ~500 k nodes (A20), not BJ's ~50 k
    assert t.depth[0] == 0 and np.all(np.diff(t.depth.astype(int)) >= 0)     # BFS order
    par, oct_ = np.nonzero(t.child >= 0)
    ch = t.child[par, oct_]
    assert np.array_equal(np.sort(ch), np.arange(1, t.n_nodes))              # every non-root node has exactly one parent
    assert np.all(t.depth[ch] == t.depth[par] + 1)
    bits = np.stack([oct_ & 1, (oct_ >> 1) & 1, (oct_ >> 2) & 1], 1)
    assert np.array_equal(t.coords[ch], t.coords[par] * 2 + bits)
    for l, d in enumerate(t.level_depth):
        sl = t.map_slot[t.depth == d]
        assert np.array_equal(sl, np.arange(t.level_slots[l]))               # slots unique and dense per used level
    assert np.all(t.map_slot[~np.isin(t.depth, t.level_depth)] == -1)
    assert [a.shape for a in cfg1_small.atlas.levels] == [(s, r, r, 8) for s, r in zip(t.level_slots, t.level_res)]
    assert all(a.dtype == np.float16 for a in cfg1_small.atlas.levels)
    a = cfg1_small.atlas.levels[3].astype(np.float64)
    assert abs(a.std() - 0.1) < 2e-3 and abs(a.mean()) < 1e-3                # N(0, std 0.1) (A18)


def test_primary_hits(cfg1_small):
    w = cfg1_small
    q = w.queries
    assert q.n == 192 * 160 and q.x.dtype == np.float32
    assert np.abs(np.linalg.norm(q.wo, axis=1) - 1).max() < 1e-6 and np.abs(np.linalg.norm(q.nrm, axis=1) - 1).max() < 1e-6
    assert (q.nrm * q.wo).sum(1).min() > -1e-6                               # wo is on the normal's hemisphere
    assert q.x.min() >= 0.03 - 1e-6 and q.x.max() <= 0.97 + 1e-6
    path = O.descend(w.tree.child, O.quantise(q.x, w.tree.max_depth), w.tree.max_depth)
    assert (path >= 0).all()                                                 # every hit lies in an existing leaf (A17)
    # the hit points lie on their surfaces
    d_sph = np.abs(np.linalg.norm(q.x[:, None, :].astype(np.float64) - w.scene.spheres[None, :, :3], axis=2) - w.scene.spheres[None, :, 3]).min(1)
    d_pl = np.minimum(np.abs(q.x.astype(np.float64) - 0.03).min(1), np.abs(q.x[:, :2].astype(np.float64) - 0.97).min(1))
    assert np.minimum(d_sph, d_pl).max() < 1e-6


def test_incoherent_sampler_and_config_shapes():
    sc = gen.make_scene("many", 0)
    assert sc.spheres.shape == (64, 4) and sc.spheres[:, 3].min() >= 0.02 and sc.spheres[:, 3].max() <= 0.07
    q = gen.incoherent_queries(sc, 20000, 0)
    assert np.array_equal(q.x[5000:6000], gen.incoherent_queries(sc, 1000, 0, first=5000).x)
    assert (q.nrm * q.wo).sum(1).min() >= -1e-6
    tree = gen.build_tree(sc, 6).set_levels([2, 4, 6], [64, 32, 16])
    path = O.descend(tree.child, O.quantise(q.x, 6), 6)
    assert (path >= 0).all()
    w0 = gen.config0()
    assert w0.tree.n_nodes == 73 and w0.tree.level_slots == [8, 64] and w0.queries.n == 4096
    assert w0.mlp.in_dim == 14 and [x.shape for x in w0.mlp.weights] == [(64, 14), (64, 64), (3, 64)]
    assert w0.atlas.levels[0].dtype == np.float32 and abs(w0.atlas.levels[1].mean()) < 0.05
    w2 = gen.scene_workload(2, width=64, height=36)
    assert w2.mlp.in_dim == 39 and w2.queries.extra.shape == (64 * 36, 1)
    assert 0.05 <= w2.queries.extra.min() and w2.queries.extra.max() <= 1.0
    std1 = w2.mlp.weights[1].astype(np.float64).std()
    assert abs(std1 - np.sqrt(2 / 64)) < 0.01                                # He-normal
