"""CPU ORACLE (numpy, float64) for the disparity predictor g_psi of the paper's Eq. 7 — the last piece of SURVEY.md §8(f) row f3.

TEST INFRASTRUCTURE ONLY (same rules as oo_oracle.py: only tests/, smoke() and bench.py's CPU legs import it; it shares
nothing with the CUDA path).

What the paper fixes (/root/reference/PAPER.md cited as P:line):
  * d^(x, w_r) = g_psi(x, w_r)                                                               Eq. 7
  * g_psi is "a compact multi-resolution hash-grid network in the style of Instant-NGP"
  * "a compact Instant-NGP-style network with 2 hidden layers of 64 neurons to predict disparity from position and
    mirror reflection direction w_r"
  * d^ is a disparity: the virtual reflected point is y = x + w_r / d^                       Eq. 8
What it does NOT give: number of grid levels, resolutions, table size, features per entry, how w_r enters the network,
the output activation.  Those are READINGS (A25-A30) and therefore **parity unpinned** as far as the
paper goes: each step below is pinned on its own (tests/test_oracle_hashgrid.py) against closed forms, a library
routine (3-D grid_sample on dense levels), brute force with python integers, and a triple-loop MLP, but no number in the
paper pins the composition.

The multi-resolution hash encoding follows the published algorithm (Mueller et al. 2022, the paper's ref. [25]), restated:
  level g has N_g intervals per axis, i.e. (N_g + 1)^3 grid vertices over [0,1]^3, and a table of T_g entries of Fh
  features;  T_g = (N_g+1)^3 if that is <= T_max (the level is DENSE: vertex (i,j,k) owns entry i + (N_g+1)(j + (N_g+1)k)),
  otherwise T_g = T_max = 2^hash_log2 and vertex (i,j,k) reads entry  ((i*1) xor (j*2654435761) xor (k*805459861)) mod T_max
  with the products taken modulo 2^32 (the spatial hash of that paper; collisions are not resolved);
  the feature at x is the trilinear interpolation of the eight vertices of the cell containing x.
Readings: resolutions N_g are DATA (the generator uses the geometric progression of that paper); x is clamped to [0,1]^3
(A16); p = x*N_g, cell c0 = min(floor(p), N_g - 1) so that x = 1 falls in the last cell with t = 1; t = p - c0.
The network input is [e_0 .. e_{G-1} | w_r] (G*Fh + 3 scalars, w_r raw as in Eq. 12); 2 hidden layers x 64, ReLU, no
biases (A10, A11); one output z and d^ = exp(z) (positive, as a disparity must be; A27).

Precision: double throughout EXCEPT the cell decision, which both sides take in fp32:
p = fl32(fl32(x) * fl32(N_g)), c0 and t = p - c0 (exact in fp32) from that p.  w_r is the fp32 sequence of
oo_oracle_full.mirror_f32.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List

import numpy as np

from . import oo_oracle as O
from . import oo_oracle_full as FO

PRIME_Y = 2654435761
PRIME_Z = 805459861


@dataclass
class HashGrid:
    res: List[int]                 # N_g, intervals per axis, coarse -> fine
    hash_log2: int                 # T_max = 2^hash_log2
    tables: List[np.ndarray]       # [T_g][Fh] (fp16 or wider; widened to double here)

    @property
    def n_features(self) -> int:
        return int(self.tables[0].shape[1])


def table_size(N: int, hash_log2: int) -> int:
    """T_g: the dense vertex count (N+1)^3 when it fits into T_max = 2^hash_log2 entries, else T_max."""
    dense = (N + 1) ** 3
    return dense if dense <= (1 << hash_log2) else (1 << hash_log2)


def is_dense(N: int, hash_log2: int) -> bool:
    return (N + 1) ** 3 <= (1 << hash_log2)


def vertex_index(i, j, k, N: int, hash_log2: int):
    """Entry of grid vertex (i, j, k), 0 <= i,j,k <= N, in level N's table (dense: row-major with i fastest; hashed: the
    xor-of-products spatial hash, products modulo 2^32)."""
    i = np.asarray(i, np.uint64)
    j = np.asarray(j, np.uint64)
    k = np.asarray(k, np.uint64)
    if is_dense(N, hash_log2):
        return (i + np.uint64(N + 1) * (j + np.uint64(N + 1) * k)).astype(np.int64)
    m32 = np.uint64(0xFFFFFFFF)
    h = (i & m32) ^ ((j * np.uint64(PRIME_Y)) & m32) ^ ((k * np.uint64(PRIME_Z)) & m32)
    return (h & np.uint64((1 << hash_log2) - 1)).astype(np.int64)


def cell_f32(x, N: int):
    """The cell decision in fp32: x clamped to [0,1] (A16); p = fl32(x * N); c0 = min(floor(p), N-1); t = p - c0 (exact).
    Returns (c0 int64 [n][3], t float64 [n][3])."""
    f = np.float32
    xc = np.minimum(np.maximum(np.asarray(x, f), f(0)), f(1))
    p = (xc * f(N)).astype(f)
    c0 = np.minimum(np.floor(p), f(N - 1)).astype(f)
    t = (p - c0).astype(f)
    return c0.astype(np.int64), t.astype(np.float64)


def encode_level(table, x, N: int, hash_log2: int):
    """Trilinear interpolation of the eight vertices of the cell containing x: sum over d in {0,1}^3 of
    prod_a (d_a ? t_a : 1 - t_a) * table[vertex_index(c0 + d)]."""
    T = np.asarray(table, np.float64)
    c0, t = cell_f32(x, N)
    out = np.zeros((c0.shape[0], T.shape[1]), np.float64)
    for dz in (0, 1):
        for dy in (0, 1):
            for dx in (0, 1):
                w = (t[:, 0] if dx else 1.0 - t[:, 0]) * (t[:, 1] if dy else 1.0 - t[:, 1]) * (t[:, 2] if dz else 1.0 - t[:, 2])
                idx = vertex_index(c0[:, 0] + dx, c0[:, 1] + dy, c0[:, 2] + dz, N, hash_log2)
                out += w[:, None] * T[idx]
    return out


def encode(grid: HashGrid, x):
    """[n][G*Fh]: the per-level features concatenated coarse to fine."""
    return np.concatenate([encode_level(grid.tables[g], x, grid.res[g], grid.hash_log2) for g in range(len(grid.res))], 1)


def network_input(grid: HashGrid, x, nrm, wo):
    """[e(x) | w_r]: the position goes through the hash grid, the mirror direction enters raw."""
    w_r = FO.mirror_f32(nrm, wo).astype(np.float64)
    return np.concatenate([encode(grid, x), w_r], 1)


def disparity(grid: HashGrid, weights, x, nrm, wo):
    """d^ = exp(z), z = the one output of the 2 x 64 ReLU network (Eq. 7)."""
    z = O.mlp(weights, network_input(grid, x, nrm, wo), "none")
    return np.exp(z[:, 0])
