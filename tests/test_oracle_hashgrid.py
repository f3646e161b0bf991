"""Pins for oracle/oo_hashgrid.py (the disparity predictor g_psi, Eq. 7): every step is
checked against something other than itself — closed forms, python-integer brute force, torch's 3-D grid_sample on dense
levels, a triple-loop MLP, and the limits Eq. 8-9 fix for the shifted direction."""
import itertools

import numpy as np
import pytest

import gen
from oracle import oo_hashgrid as HG
from oracle import oo_oracle_full as FO

torch = pytest.importorskip("torch")


def _pts(n, seed):
    return np.random.default_rng(seed).random((n, 3)).astype(np.float32)


# ------------------------------------------------------------------------------------------------ table layout


def test_table_size_and_density_rule():
    assert HG.table_size(16, 17) == 17 ** 3 and HG.is_dense(16, 17)
    assert HG.table_size(43, 17) == 44 ** 3 and HG.is_dense(43, 17)          # 85,184 <= 131,072
    assert HG.table_size(50, 17) == 1 << 17 and not HG.is_dense(50, 17)      # 51^3 = 132,651 > 131,072
    assert HG.table_size(1, 3) == 8 and HG.is_dense(1, 3)                    # exactly full still counts as dense


def test_dense_index_is_row_major_i_fastest():
    N = 5
    seen = set()
    for k, j, i in itertools.product(range(N + 1), repeat=3):
        idx = int(HG.vertex_index(i, j, k, N, 17))
        assert idx == i + 6 * j + 36 * k
        seen.add(idx)
    assert seen == set(range(216))


def test_hash_values_by_python_integers():
    """The spatial hash of the paper's ref. [25]: xor of per-axis products (modulo 2^32) with primes 1, 2654435761,
    805459861, reduced modulo the table size; here recomputed with unbounded python integers."""
    lg = 12
    T = 1 << lg
    assert int(HG.vertex_index(1, 0, 0, 100, lg)) == 1
    assert int(HG.vertex_index(0, 1, 0, 100, lg)) == 2654435761 % T == 0x9B1     # 2654435761 = 0x9E3779B1
    assert int(HG.vertex_index(0, 0, 1, 100, lg)) == 805459861 % T == 0x795          # 805459861 = 0x30025795
    assert int(HG.vertex_index(1, 1, 1, 100, lg)) == (1 ^ 2654435761 ^ 805459861) % T
    r = np.random.default_rng(1)
    for i, j, k in r.integers(0, 513, size=(200, 3)):
        want = ((int(i) & 0xFFFFFFFF) ^ ((int(j) * 2654435761) & 0xFFFFFFFF) ^ ((int(k) * 805459861) & 0xFFFFFFFF)) % (1 << 17)
        assert int(HG.vertex_index(i, j, k, 512, 17)) == want


def test_hashed_index_vectorised_equals_scalar():
    ijk = np.random.default_rng(2).integers(0, 313, size=(1000, 3))
    v = HG.vertex_index(ijk[:, 0], ijk[:, 1], ijk[:, 2], 312, 17)
    for a in range(0, 1000, 37):
        assert v[a] == int(HG.vertex_index(int(ijk[a, 0]), int(ijk[a, 1]), int(ijk[a, 2]), 312, 17))
    assert v.min() >= 0 and v.max() < (1 << 17)


# ------------------------------------------------------------------------------------------------ cell decision


def test_cell_and_fraction_closed_form_and_edges():
    x = np.array([[0.0, 0.5, 1.0], [0.25, 0.999999, 0.1], [-0.5, 1.5, 0.3]], np.float32)
    c0, t = HG.cell_f32(x, 16)
    assert c0.tolist() == [[0, 8, 15], [4, 15, 1], [0, 15, 4]]              # x = 1 (and beyond: clamped) -> last cell ...
    assert t[0].tolist() == [0.0, 0.0, 1.0] and t[2, 1] == 1.0               # ... with t = 1
    assert abs(t[1, 2] - (np.float32(0.1) * np.float32(16) - 1)) < 1e-6
    # power-of-two N: the fp32 product is exact, so the fp32 decision equals the exact one
    xs = _pts(20000, 3)
    c0, t = HG.cell_f32(xs, 64)
    p = xs.astype(np.float64) * 64
    assert np.array_equal(c0, np.floor(p).astype(np.int64)) and np.abs(t - (p - c0)).max() == 0.0
    # any N: within one fp32 rounding of the exact position, and the reconstructed p = c0 + t is that fp32 product
    for N in (26, 43, 190, 312):
        c0, t = HG.cell_f32(xs, N)
        p32 = (xs * np.float32(N)).astype(np.float32)
        assert np.array_equal((c0 + t).astype(np.float32), p32)
        assert np.abs((c0 + t) - xs.astype(np.float64) * N).max() <= N * 2.0 ** -24
        assert c0.min() >= 0 and c0.max() <= N - 1 and t.min() >= 0.0 and t.max() <= 1.0


# ------------------------------------------------------------------------------------------------ interpolation


def test_constant_table_gives_the_constant():
    for N, lg in ((16, 17), (190, 17)):
        T = np.full((HG.table_size(N, lg), 2), [0.75, -1.5])
        e = HG.encode_level(T, _pts(500, 4), N, lg)
        assert np.abs(e - [0.75, -1.5]).max() < 1e-15


def test_dense_level_reproduces_linear_fields_exactly():
    """Trilinear interpolation over grid vertices reproduces any affine function of position."""
    N, lg = 26, 17
    k, j, i = np.meshgrid(np.arange(N + 1), np.arange(N + 1), np.arange(N + 1), indexing="ij")
    a = np.array([0.3, -1.1, 2.0, 0.25])
    T = np.stack([a[0] * i / N + a[1] * j / N + a[2] * k / N + a[3], (i + j + k) / N], -1).reshape(-1, 2)   # entry i + (N+1)(j + (N+1)k)
    x = _pts(2000, 5)
    c0, t = HG.cell_f32(x, N)
    xe = (c0 + t) / N                                    # the position the fp32 cell decision stands for
    e = HG.encode_level(T, x, N, lg)
    assert np.abs(e[:, 0] - (xe @ a[:3] + a[3])).max() < 1e-13
    assert np.abs(e[:, 1] - xe.sum(1)).max() < 1e-13
    assert np.abs(xe - x).max() < 2.0 ** -23


def test_dense_level_equals_grid_sample_3d():
    """torch's grid_sample (trilinear, align_corners=True) puts the corners of [-1,1]^3 on the first and last vertex:
    exactly the vertex grid of a dense level."""
    N, lg = 16, 17
    r = np.random.default_rng(6)
    T = r.normal(size=((N + 1) ** 3, 2))
    x = _pts(3000, 7)
    e = HG.encode_level(T, x, N, lg)
    vol = torch.from_numpy(T.reshape(N + 1, N + 1, N + 1, 2)).permute(3, 0, 1, 2)[None]          # [1][C][D=k][H=j][W=i]
    grid = torch.from_numpy(x.astype(np.float64) * 2 - 1).reshape(1, -1, 1, 1, 3)                 # (x -> W, y -> H, z -> D)
    ref = torch.nn.functional.grid_sample(vol, grid, mode="bilinear", align_corners=True)[0, :, :, 0, 0].T.numpy()
    assert np.abs(e - ref).max() < 1e-12


def test_hashed_level_by_brute_force():
    """A hashed level, evaluated point by point with python scalars and a dictionary of hashed vertices."""
    N, lg = 70, 10
    r = np.random.default_rng(8)
    T = r.normal(size=(1 << lg, 2))
    x = _pts(60, 9)
    e = HG.encode_level(T, x, N, lg)
    for q in range(60):
        p = [float(np.float32(x[q, a]) * np.float32(N)) for a in range(3)]
        c = [min(int(np.floor(v)), N - 1) for v in p]
        t = [p[a] - c[a] for a in range(3)]
        acc = np.zeros(2)
        for dx, dy, dz in itertools.product((0, 1), repeat=3):
            i, j, k = c[0] + dx, c[1] + dy, c[2] + dz
            h = (i ^ ((j * 2654435761) & 0xFFFFFFFF) ^ ((k * 805459861) & 0xFFFFFFFF)) % (1 << lg)
            w = (t[0] if dx else 1 - t[0]) * (t[1] if dy else 1 - t[1]) * (t[2] if dz else 1 - t[2])
            acc += w * T[h]
        assert np.abs(acc - e[q]).max() < 1e-13


def test_at_a_vertex_the_feature_is_that_vertex_entry_and_collisions_alias():
    N, lg = 128, 8                                       # power-of-two N: vertex positions i/N are exact; 256 entries -> many collisions
    T = np.random.default_rng(10).normal(size=(1 << lg, 2))
    ijk = np.array([[3, 77, 100], [0, 0, 0], [128, 128, 128], [64, 1, 127]])
    e = HG.encode_level(T, (ijk / N).astype(np.float32), N, lg)
    for a, (i, j, k) in enumerate(ijk):
        assert np.array_equal(e[a], T[int(HG.vertex_index(i, j, k, N, lg))])
    # two different vertices with the same hash read the same entry (collisions are not resolved)
    seen = {}
    for i, j, k in itertools.product(range(12), repeat=3):
        seen.setdefault(int(HG.vertex_index(i, j, k, N, lg)), []).append((i, j, k))
    a, b = next(v for v in seen.values() if len(v) >= 2)[:2]
    ea = HG.encode_level(T, (np.array([a]) / N).astype(np.float32), N, lg)
    eb = HG.encode_level(T, (np.array([b]) / N).astype(np.float32), N, lg)
    assert a != b and np.array_equal(ea, eb)


def test_feature_is_continuous_across_cell_faces():
    d = gen.make_disparity_net(0, n_levels=4, n_min=8, n_max=64, hash_log2=12)
    grid = HG.HashGrid(d.res, d.hash_log2, d.tables)
    r = np.random.default_rng(11)
    x = r.random((500, 3))
    x[:, 0] = r.integers(1, 8, 500) / 8.0                # on a face of every level's grid? only of level 0 (N = 8) for sure
    lo = HG.encode(grid, (x - [1e-6, 0, 0]).astype(np.float32))
    hi = HG.encode(grid, (x + [1e-6, 0, 0]).astype(np.float32))
    assert np.abs(lo - hi).max() < 1e-3                  # |grad| <= 2 * max|entry| * N_max ~ 300, times 2e-6 apart


def test_encode_concatenates_levels_coarse_to_fine():
    d = gen.make_disparity_net(1, n_levels=3, n_min=4, n_max=40, hash_log2=10)
    grid = HG.HashGrid(d.res, d.hash_log2, d.tables)
    assert grid.n_features == 2 and d.res == [4, 12, 40]
    x = _pts(50, 12)
    e = HG.encode(grid, x)
    assert e.shape == (50, 6)
    for g in range(3):
        assert np.array_equal(e[:, 2 * g:2 * g + 2], HG.encode_level(d.tables[g], x, d.res[g], d.hash_log2))


# ------------------------------------------------------------------------------------------------ network


def test_network_input_layout_and_mlp_by_triple_loop():
    d = gen.make_disparity_net(2, n_levels=3, n_min=4, n_max=40, hash_log2=10)
    grid = HG.HashGrid(d.res, d.hash_log2, d.tables)
    q = gen.random_queries(40, 3)
    inp = HG.network_input(grid, q.x, q.nrm, q.wo)
    assert inp.shape == (40, 9)
    assert np.array_equal(inp[:, :6], HG.encode(grid, q.x))
    n, w = q.nrm.astype(np.float64), q.wo.astype(np.float64)
    assert np.abs(inp[:, 6:] - (2 * (n * w).sum(1, keepdims=True) * n - w)).max() < 1e-6       # w_r = 2(n.wo)n - wo
    got = HG.disparity(grid, d.weights, q.x, q.nrm, q.wo)
    for a in range(0, 40, 7):
        act = [float(v) for v in inp[a]]
        for W in d.weights[:-1]:
            act = [max(0.0, sum(float(W[o, i]) * act[i] for i in range(W.shape[1]))) for o in range(W.shape[0])]
        z = sum(float(d.weights[-1][0, i]) * act[i] for i in range(64))
        assert abs(np.exp(z) - got[a]) <= 1e-12 * np.exp(z)
    assert (got > 0).all()


def test_zero_output_layer_gives_unit_disparity():
    d = gen.make_disparity_net(3, n_levels=2, n_min=4, n_max=8, hash_log2=10)
    d.weights[-1][:] = 0
    q = gen.random_queries(10, 4)
    assert np.array_equal(HG.disparity(HG.HashGrid(d.res, d.hash_log2, d.tables), d.weights, q.x, q.nrm, q.wo), np.ones(10))


# ------------------------------------------------------------------------------------------------ Eq. 8-9 limits


def test_shifted_direction_limits_of_eq_9():
    """d^ -> 0 (reflected point at infinity): w~_j = w_r for every cell; d^ -> infinity: w~_j points from the cell centre
    to x.  Both follow from Eq. 8-9 and pin how d^ enters the lookup."""
    q = gen.random_queries(200, 5)
    w_r = FO.mirror_f32(q.nrm, q.wo)
    c = np.full((200, 3), 0.5, np.float32)
    near0 = FO.shifted_f32(q.x, c, np.full(200, 1e-12, np.float32), w_r).astype(np.float64)
    assert np.abs(near0 - w_r).max() < 1e-6
    far = FO.shifted_f32(q.x, c, np.full(200, 1e9, np.float32), w_r).astype(np.float64)
    far /= np.linalg.norm(far, axis=1, keepdims=True)
    want = (q.x - c).astype(np.float64)
    want /= np.linalg.norm(want, axis=1, keepdims=True)
    assert np.abs(far - want).max() < 1e-6
    # and the literal Eq. 8-9 (y = x + w_r/d^, normalised) agrees with the un-normalised fp32 form up to scale
    d = gen.disparity(200, 6)
    a = FO.shifted_f32(q.x, c, d, w_r).astype(np.float64)
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    assert np.abs(a - FO.shifted_f64(q.x, c, d, w_r)).max() < 1e-5
