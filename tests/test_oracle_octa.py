"""Pins for the oracle's octahedral projection, texel lookup, wrap and bilinear interpolation (O3-O6).

Each test ties the oracle to something other than itself: hand-evaluated values of Eq. 4-5 (tests/golden), closed
forms, invariants stated by the paper (continuity across the spherical domain), a library special case
(torch grid_sample), brute-force definitions.  A dropped term, wrong sign, swapped axis or wrong wrap fails one."""
import os

import numpy as np
import pytest

from oracle import oo_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            out.append([float(t) for t in line.replace("|", " ").replace("->", " ").split()])
    return out


def _unit(n, seed):
    rng = np.random.default_rng(seed)
    w = rng.normal(size=(n, 3))
    return w / np.linalg.norm(w, axis=1, keepdims=True)


def test_fixed_images_of_the_axes():
    # Eq. 4-5, sign(0)=+1 (A1): +x->(1,0) -x->(-1,0) +y->(0,1) -y->(0,-1) +z->(0,0) -z->(1,1)
    w = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], float)
    u = O.octa_encode(w)
    assert np.array_equal(u, np.array([[1, 0], [-1, 0], [0, 1], [0, -1], [0, 0], [1, 1]], float))
    v = (u + 1) / 2
    assert np.array_equal(v, np.array([[1, .5], [0, .5], [.5, 1], [.5, 0], [.5, .5], [1, 1]]))


def test_golden_worked_examples():
    for r in _rows("octa_examples.txt"):
        w = np.array([r[0:3]])
        u = O.octa_encode(w)[0]
        assert np.allclose(u, r[3:5], atol=1e-15)
        s = O.sample_coord(u, 8)
        assert np.allclose(s, r[5:7], atol=1e-14)
        i0, j0 = O.texel_base_f32(w, 8)
        assert (int(i0[0]), int(j0[0])) == (int(r[7]), int(r[8]))
        fx, fy = s[0] - i0[0], s[1] - j0[0]
        wts = [(1 - fx) * (1 - fy), fx * (1 - fy), (1 - fx) * fy, fx * fy]
        assert np.allclose(wts, r[9:13], atol=1e-14)
        # and through dir_interp itself: a map that is 1 at one texel returns that tap's weight
        for k, (a, b) in enumerate([(0, 0), (1, 0), (0, 1), (1, 1)]):
            ii, jj = O.wrap(np.array([int(r[7]) + a]), np.array([int(r[8]) + b]), 8)
            T = np.zeros((1, 8, 8, 1))
            T[0, jj[0], ii[0], 0] = 1.0
            h, _, _ = O.dir_interp(T, np.array([0]), w.astype(np.float32), 8)
            same = sum(1 for (a2, b2) in [(0, 0), (1, 0), (0, 1), (1, 1)]
                       if tuple(x[0] for x in O.wrap(np.array([int(r[7]) + a2]), np.array([int(r[8]) + b2]), 8)) == (ii[0], jj[0]))
            expect = sum(r[9 + k2] for k2, (a2, b2) in enumerate([(0, 0), (1, 0), (0, 1), (1, 1)])
                         if tuple(x[0] for x in O.wrap(np.array([int(r[7]) + a2]), np.array([int(r[8]) + b2]), 8)) == (ii[0], jj[0]))
            assert same >= 1 and abs(h[0, 0] - expect) < 1e-6


def test_golden_wrapped_taps():
    for r in _rows("wrap_taps.txt"):
        i, j = O.wrap(np.array([int(r[0])]), np.array([int(r[1])]), 8)
        assert (i[0], j[0]) == (int(r[2]), int(r[3]))


def test_round_trip_and_range():
    w = _unit(20000, 1)
    u = O.octa_encode(w)
    assert u.min() >= -1 and u.max() <= 1
    # |ux|+|uy| <= 1  <=>  z >= 0 (upper hemisphere is the inner diamond)
    l1 = np.abs(u).sum(1)
    assert np.all((l1 <= 1 + 1e-15) == (w[:, 2] >= 0) | (np.abs(l1 - 1) < 1e-12))
    assert np.abs(O.octa_decode(u) - w).max() < 1e-14
    rng = np.random.default_rng(2)
    uu = rng.uniform(-1, 1, size=(20000, 2))
    assert np.abs(O.octa_encode(O.octa_decode(uu)) - uu).max() < 1e-14
    # Eq. 4 is scale invariant (A22)
    assert np.abs(O.octa_encode(w * 3.7) - u).max() < 1e-15


def test_octa_is_not_axis_swapped():
    # u_x follows w_x and u_y follows w_y on the upper hemisphere (Eq. 4)
    u = O.octa_encode(np.array([[0.6, 0.0, 0.8], [0.0, 0.6, 0.8]]))
    assert u[0, 0] > 0 and u[0, 1] == 0 and u[1, 0] == 0 and u[1, 1] > 0


def _wrap_geometric(i, j, R):
    """Independent derivation in continuous coordinates: texel centre -> u; if |u_x| > 1 point-reflect about
    (sign, 0): (u_x, u_y) -> (2 sign - u_x, -u_y); same for y; back to the texel index."""
    ux, uy = (i + 0.5) / R * 2 - 1, (j + 0.5) / R * 2 - 1
    if abs(ux) > 1:
        ux, uy = 2 * np.sign(ux) - ux, -uy
    if abs(uy) > 1:
        ux, uy = -ux, 2 * np.sign(uy) - uy
    return int(round((ux + 1) / 2 * R - 0.5)), int(round((uy + 1) / 2 * R - 0.5))


@pytest.mark.parametrize("R", [2, 4, 8, 16])
def test_wrap_exhaustive_and_order_independent(R):
    for i in range(-1, R + 1):
        for j in range(-1, R + 1):
            a = O.wrap(np.array([i]), np.array([j]), R)
            assert (a[0][0], a[1][0]) == _wrap_geometric(i, j, R)
            # I5: y-rule first then x-rule gives the same texel
            jj, ii = O.wrap(np.array([j]), np.array([i]), R)   # wrap is symmetric under swapping the roles of the axes
            assert (ii[0], jj[0]) == (a[0][0], a[1][0])
            if 0 <= i < R and 0 <= j < R:
                assert (a[0][0], a[1][0]) == (i, j)
    # doubly-outside corner taps land on the diagonally opposite corner
    for (i, j), e in {(-1, -1): (R - 1, R - 1), (R, R): (0, 0), (-1, R): (R - 1, 0), (R, -1): (0, R - 1)}.items():
        a = O.wrap(np.array([i]), np.array([j]), R)
        assert (a[0][0], a[1][0]) == e


def test_wrapped_tap_is_the_same_direction_on_the_sphere():
    """The geometric content of the wrap, through octa_decode only: a point just outside the square, reflected about
    the edge midpoint, decodes to a direction close to the decode of the point mirrored back across the edge — i.e.
    the reflected point is the *neighbour on the sphere* of the edge point, not an arbitrary texel."""
    rng = np.random.default_rng(5)
    t = rng.uniform(-1, 1, 200)
    eps = 1e-6
    inside = np.stack([np.full_like(t, 1 - eps), t], 1)            # just inside the edge u_x = 1
    cont = np.stack([np.full_like(t, 1 - eps), -t], 1)             # image of (1+eps, t) under the point reflection
    edge_a = O.octa_decode(np.stack([np.ones_like(t), t], 1))
    edge_b = O.octa_decode(np.stack([np.ones_like(t), -t], 1))
    assert np.abs(edge_a - edge_b).max() < 1e-12                   # I1: (1,t) and (1,-t) are the same direction
    assert np.abs(O.octa_decode(inside) - edge_a).max() < 1e-5
    assert np.abs(O.octa_decode(cont) - edge_a).max() < 1e-5       # both sides of the seam are neighbours on the sphere


@pytest.mark.parametrize("R", [4, 8, 32])
def test_constant_and_linear_fields_reproduced_exactly(R):
    w = _unit(5000, 3).astype(np.float32)
    slot = np.zeros(len(w), np.int64)
    T = np.full((1, R, R, 3), 0.731)
    h, _, _ = O.dir_interp(T, slot, w, R)
    assert np.abs(h - 0.731).max() < 1e-15                         # I3 (weights sum to 1)
    jj, ii = np.meshgrid(np.arange(R), np.arange(R), indexing="ij")
    al, be, ga = 0.3, -0.11, 0.07
    T = (al + be * ii + ga * jj)[None, :, :, None].astype(np.float64)   # T[slot][j][i]
    h, i0, j0 = O.dir_interp(T, slot, w, R)
    s = O.sample_coord(O.octa_encode(w.astype(np.float64)), R)
    interior = (i0 >= 0) & (i0 < R - 1) & (j0 >= 0) & (j0 < R - 1)
    assert interior.sum() > 100
    assert np.abs(h[interior, 0] - (al + be * s[interior, 0] + ga * s[interior, 1])).max() < 1e-13   # I4


@pytest.mark.parametrize("R", [4, 16])
def test_library_special_case_grid_sample(R):
    """Interior samples equal torch.nn.functional.grid_sample(bilinear, align_corners=False): that convention puts
    texel centres at (i+1/2)/R over [-1,1], i.e. exactly s = (u+1)/2*R - 1/2 with x <-> i (width) and y <-> j (height)."""
    import torch
    rng = np.random.default_rng(7)
    T = rng.normal(size=(1, R, R, 5))
    w = _unit(4000, 8).astype(np.float32)
    h, i0, j0 = O.dir_interp(T, np.zeros(len(w), np.int64), w, R)
    u = O.octa_encode(w.astype(np.float64))
    img = torch.from_numpy(T[0]).permute(2, 0, 1)[None]                     # [1][F][H=j][W=i]
    grid = torch.from_numpy(u)[None, None]                                  # [1][1][N][2] = (x, y)
    ref = torch.nn.functional.grid_sample(img, grid, mode="bilinear", padding_mode="zeros", align_corners=False)
    ref = ref[0, :, 0, :].T.numpy()
    interior = (i0 >= 0) & (i0 < R - 1) & (j0 >= 0) & (j0 < R - 1)
    assert interior.sum() > 100
    assert np.abs(h[interior] - ref[interior]).max() < 1e-12


def _interp_at_u(T, u, R):
    """Interpolant evaluated at map coordinates u (test helper, double only, via decode -> direction)."""
    w = O.octa_decode(u)
    h, _, _ = O.dir_interp(T, np.zeros(len(w), np.int64), w.astype(np.float32), R)
    return h


@pytest.mark.parametrize("R", [4, 8])
def test_continuity_across_the_spherical_domain(R):
    """"the interpolation is continuous across the spherical domain".  With a random map, (a) the value just
    on either side of every outer edge agrees (seam continuity), (b) edge-identified points give equal values (I1),
    (c) all four corners (= -z) give the mean of the four corner texels (I2), (d) the interpolant is Lipschitz over
    random nearby direction pairs anywhere on the sphere.  Clamp-to-edge or a plain mirror wrap fails (a)/(b)."""
    rng = np.random.default_rng(11)
    T = rng.normal(size=(1, R, R, 2))
    a = rng.uniform(0.02, 0.98, 300)
    one, zero = np.ones_like(a), np.zeros_like(a)
    v_pairs = [(np.stack([one, a], 1), np.stack([one, 1 - a], 1)), (np.stack([zero, a], 1), np.stack([zero, 1 - a], 1)),
               (np.stack([a, one], 1), np.stack([1 - a, one], 1)), (np.stack([a, zero], 1), np.stack([1 - a, zero], 1))]
    for va, vb in v_pairs:                                        # (b) I1
        ha, hb = _interp_at_u(T, 2 * va - 1, R), _interp_at_u(T, 2 * vb - 1, R)
        assert np.abs(ha - hb).max() < 1e-5
    corners = np.array([[0, 0], [1, 0], [0, 1], [1, 1]], float)   # (c) I2
    hc = _interp_at_u(T, 2 * corners - 1, R)
    mean4 = 0.25 * (T[0, 0, 0] + T[0, 0, R - 1] + T[0, R - 1, 0] + T[0, R - 1, R - 1])
    assert np.abs(hc - mean4).max() < 1e-5
    # (a)+(d): directions straddling the seams x=0 / y=0 of the lower hemisphere and random nearby pairs
    w = _unit(20000, 12)
    w[:5000, 0] = np.abs(w[:5000, 0]) * 1e-7                      # hug the meridian x = 0 (a seam when z < 0)
    w[:5000, 2] = -np.abs(w[:5000, 2])
    w[5000:10000, 1] = np.abs(w[5000:10000, 1]) * 1e-7
    w[5000:10000, 2] = -np.abs(w[5000:10000, 2])
    w /= np.linalg.norm(w, axis=1, keepdims=True)
    d = rng.normal(size=w.shape) * 1e-4
    d[:5000, 0] = -2e-7                                           # step across the seam
    d[5000:10000, 1] = -2e-7
    w2 = w + d
    w2 /= np.linalg.norm(w2, axis=1, keepdims=True)
    zero_slot = np.zeros(len(w), np.int64)
    h1, _, _ = O.dir_interp(T, zero_slot, w.astype(np.float32), R)
    h2, _, _ = O.dir_interp(T, zero_slot, w2.astype(np.float32), R)
    dist = np.linalg.norm(w.astype(np.float32).astype(np.float64) - w2.astype(np.float32).astype(np.float64), axis=1)
    # |grad| of a bilinear map in u is <= 2*R*max|dT| ~ R*8 and |du/dw| <= ~3 near the poles of the L1 normalisation
    lip = np.abs(h1 - h2).max(1) / np.maximum(dist, 1e-9)
    assert lip.max() < 60 * R, lip.max()
    assert np.abs(h1[:10000] - h2[:10000]).max() < 5e-3           # across the seam: O(|dw| = 1e-4), not O(1)


def test_clamp_to_edge_would_fail_the_seam_test():
    """Sanity of the pin itself: replace the wrap by clamp-to-edge and (b) must break (so the test has teeth)."""
    R = 8
    rng = np.random.default_rng(13)
    T = rng.normal(size=(1, R, R, 1))
    a = rng.uniform(0.05, 0.45, 50)
    va, vb = np.stack([np.ones_like(a), a], 1), np.stack([np.ones_like(a), 1 - a], 1)

    def clamp_interp(v):
        s = v * R - 0.5
        i0, j0 = np.floor(s[:, 0]).astype(int), np.floor(s[:, 1]).astype(int)
        fx, fy = s[:, 0] - i0, s[:, 1] - j0
        out = 0
        for b in (0, 1):
            for aa in (0, 1):
                out = out + (fx if aa else 1 - fx) * (fy if b else 1 - fy) * T[0, np.clip(j0 + b, 0, R - 1), np.clip(i0 + aa, 0, R - 1), 0]
        return out
    assert np.abs(clamp_interp(va) - clamp_interp(vb)).max() > 0.1


def test_fp32_index_contract_vs_double():
    """The fp32 base texel is in range without clamping, agrees with the double decision except for a ~1e-6
    fraction of directions, and at a disagreement the interpolated value is unaffected."""
    w = _unit(400000, 17).astype(np.float32)
    rng = np.random.default_rng(18)
    for R in (4, 16, 64):
        i0, j0 = O.texel_base_f32(w, R)
        assert i0.min() >= -1 and i0.max() <= R - 1 and j0.min() >= -1 and j0.max() <= R - 1
        i1, j1 = O.texel_base_f64(w, R)
        bad = (i0 != i1) | (j0 != j1)
        assert bad.mean() < 1e-4
        assert np.abs(i0 - i1).max() <= 1 and np.abs(j0 - j1).max() <= 1
    # axis-aligned and exactly-on-texel-boundary directions: fp32 decision as hand computed
    w = np.array([[1, 0, 0], [0, 0, -1], [0, 0, 1], [-1, 0, 0], [0, -1, 0]], np.float32)
    i0, j0 = O.texel_base_f32(w, 8)
    assert list(zip(i0, j0)) == [(7, 3), (7, 7), (3, 3), (-1, 3), (3, -1)]


def test_negative_zero_and_sign_convention():
    # sgn(-0.0) = +1 (A1): w = (-0, 0, -1) folds to u = (+1, +1), not (-1, +1)
    u = O.octa_encode(np.array([[-0.0, 0.0, -1.0]]))
    assert np.array_equal(u, [[1.0, 1.0]])
    i0, j0 = O.texel_base_f32(np.array([[-0.0, 0.0, -1.0]], np.float32), 8)
    assert (i0[0], j0[0]) == (7, 7)
