"""Seeded synthetic input generators for the OctaOctree query path (BASELINE.json configs 0-4).

Inputs only: random numbers, analytic scenes, octrees, atlases, MLP weights, camera rays.  None of the
method's arithmetic lives here (no descent, no octahedral map, no interpolation, no MLP), so this
module may serve both the CPU oracle (``oracle/``) and the CUDA path (``paper_2606_08469_b200/``),
which share nothing else.  The heavy parts are in ``oo_gen.c`` (gcc, OpenMP), bound with ctypes.

Recipe and citations: DESIGN.md "Input recipe" (BASELINE.json ``configs``).
Everything is generated on the host once, rounded to its storage type (fp32 queries, fp16/fp32
texels, fp16 weights); both sides then read the very same bytes.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oo_gen.c")
_LIB = os.path.join(_HERE, "liboo_gen.so")

# RNG stream ids (SURVEY.md §8(d) "Common generator rules")
STREAM_ATLAS = 100      # + level
STREAM_WEIGHTS = 200    # + layer
STREAM_POS, STREAM_NRM, STREAM_DIR, STREAM_ROUGH = 3, 4, 5, 6
STREAM_SCENE, STREAM_CAMERA, STREAM_INCOH, STREAM_SHUFFLE = 7, 8, 9, 10
STREAM_DISPARITY, STREAM_ALBEDO = 11, 12
STREAM_HASHGRID = 300   # + level
STREAM_DISP_WEIGHTS = 400   # + layer


def build_lib(force: bool = False) -> str:
    """Compile oo_gen.c -> liboo_gen.so (in-tree) if missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Scene(C.Structure):
    _fields_ = [("n_spheres", C.c_int32), ("spheres", C.POINTER(C.c_double)), ("lo", C.c_double),
                ("hi", C.c_double), ("eps", C.c_double)]


class _TreeOut(C.Structure):
    _fields_ = [("n_nodes", C.c_uint32), ("child", C.POINTER(C.c_int32)), ("depth", C.POINTER(C.c_uint8)),
                ("coords", C.POINTER(C.c_uint32)), ("depth_first", C.c_uint32 * 34)]


class _Camera(C.Structure):
    _fields_ = [("eye", C.c_double * 3), ("look", C.c_double * 3), ("up", C.c_double * 3),
                ("vfov_deg", C.c_double), ("width", C.c_uint32), ("height", C.c_uint32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build_lib())
        u64, dbl, vp = C.c_uint64, C.c_double, C.c_void_p
        L.oo_gen_u01.argtypes = [u64, u64, u64, u64, vp]
        L.oo_gen_normal.argtypes = [u64, u64, u64, u64, vp]
        L.oo_gen_normal_f16.argtypes = [u64, u64, u64, u64, dbl, vp]
        L.oo_gen_uniform_f32.argtypes = [u64, u64, u64, u64, dbl, dbl, vp]
        L.oo_gen_f64_to_f16.argtypes = [vp, u64, vp]
        L.oo_gen_normals_and_dirs.argtypes = [u64, u64, u64, u64, u64, vp, vp]
        L.oo_gen_free.argtypes = [vp]
        L.oo_gen_build_tree.argtypes = [C.POINTER(_Scene), C.c_uint32, C.c_int, C.POINTER(_TreeOut)]
        L.oo_gen_build_tree.restype = C.c_int
        L.oo_gen_raycast.argtypes = [C.POINTER(_Scene), C.POINTER(_Camera), C.c_uint32, C.c_uint32, vp, vp, vp, vp]
        L.oo_gen_raycast.restype = C.c_uint64
        L.oo_gen_incoherent.argtypes = [C.POINTER(_Scene), u64, u64, u64, u64, vp, vp, vp]
        for f in (L.oo_gen_u01, L.oo_gen_normal, L.oo_gen_normal_f16, L.oo_gen_uniform_f32, L.oo_gen_f64_to_f16,
                  L.oo_gen_normals_and_dirs, L.oo_gen_free, L.oo_gen_incoherent):
            f.restype = None
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


# ----------------------------------------------------------------------------------------- raw RNG

def u01(seed: int, stream: int, n: int, first: int = 0) -> np.ndarray:
    out = np.empty(n, np.float64)
    lib().oo_gen_u01(seed, stream, first, n, _ptr(out))
    return out


def normal(seed: int, stream: int, n: int, first: int = 0) -> np.ndarray:
    out = np.empty(n, np.float64)
    lib().oo_gen_normal(seed, stream, first, n, _ptr(out))
    return out


def normal_f16(seed: int, stream: int, n: int, std: float, first: int = 0, out: Optional[np.ndarray] = None) -> np.ndarray:
    if out is None:
        out = np.empty(n, np.float16)
    assert out.dtype == np.float16 and out.size == n and out.flags.c_contiguous
    lib().oo_gen_normal_f16(seed, stream, first, n, float(std), _ptr(out))
    return out


def uniform_f32(seed: int, stream: int, n: int, lo: float, hi: float, first: int = 0) -> np.ndarray:
    out = np.empty(n, np.float32)
    lib().oo_gen_uniform_f32(seed, stream, first, n, float(lo), float(hi), _ptr(out))
    return out


def f64_to_f16(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a, np.float64)
    out = np.empty(a.shape, np.float16)
    lib().oo_gen_f64_to_f16(_ptr(a), a.size, _ptr(out))
    return out


# ----------------------------------------------------------------------------------------- records

@dataclass
class Scene:
    spheres: np.ndarray            # [n][4] float64 (cx, cy, cz, r)
    lo: float = 0.03
    hi: float = 0.97
    eps: float = 1e-5

    def _c(self):
        self._sph = np.ascontiguousarray(self.spheres, np.float64).reshape(-1, 4)
        return _Scene(len(self._sph), self._sph.ctypes.data_as(C.POINTER(C.c_double)), self.lo, self.hi, self.eps)


@dataclass
class Camera:
    eye: np.ndarray
    look: np.ndarray
    width: int
    height: int
    vfov_deg: float = 60.0
    up: tuple = (0.0, 1.0, 0.0)

    def _c(self):
        return _Camera((C.c_double * 3)(*self.eye), (C.c_double * 3)(*self.look), (C.c_double * 3)(*self.up),
                       self.vfov_deg, self.width, self.height)


@dataclass
class Tree:
    """Logical octree. Node 0 = root (depth 0, cube [0,1]^3); octant o = bx | by<<1 | bz<<2."""
    max_depth: int
    child: np.ndarray              # [n_nodes][8] int32, -1 = absent
    depth: np.ndarray              # [n_nodes] uint8
    coords: np.ndarray             # [n_nodes][3] uint32 integer cell coordinates at the node's depth
    depth_first: np.ndarray        # [max_depth+2] first node id of each depth
    level_depth: List[int] = field(default_factory=list)   # used levels, coarse -> fine
    level_res: List[int] = field(default_factory=list)     # R_l
    map_slot: Optional[np.ndarray] = None                  # [n_nodes] int32, -1 if depth not used
    level_slots: List[int] = field(default_factory=list)

    @property
    def n_nodes(self) -> int:
        return int(self.child.shape[0])

    def set_levels(self, level_depth, level_res):
        self.level_depth = [int(d) for d in level_depth]
        self.level_res = [int(r) for r in level_res]
        self.map_slot = np.full(self.n_nodes, -1, np.int32)
        self.level_slots = []
        for d in self.level_depth:
            a, b = int(self.depth_first[d]), int(self.depth_first[d + 1])
            self.map_slot[a:b] = np.arange(b - a, dtype=np.int32)
            self.level_slots.append(b - a)
        return self


@dataclass
class Atlas:
    F: int
    dtype: str                     # "f16" | "f32"
    levels: List[np.ndarray]       # per used level [slots][R][R][F], row j (v_y) major, i (v_x) minor

    @property
    def nbytes(self) -> int:
        return sum(a.nbytes for a in self.levels)


@dataclass
class MLP:
    in_dim: int
    width: int
    n_hidden: int
    out_dim: int
    weights: List[np.ndarray]      # fp16, row-major [out][in]: [width][in_dim], [width][width]..., [out_dim][width]
    out_act: str = "exp"           # "exp" | "none"


@dataclass
class Queries:
    x: np.ndarray                  # [N][3] float32
    nrm: np.ndarray
    wo: np.ndarray
    extra: Optional[np.ndarray] = None   # [N][E] float32

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    def take(self, idx) -> "Queries":
        return Queries(np.ascontiguousarray(self.x[idx]), np.ascontiguousarray(self.nrm[idx]),
                       np.ascontiguousarray(self.wo[idx]),
                       None if self.extra is None else np.ascontiguousarray(self.extra[idx]))


@dataclass
class Workload:
    name: str
    tree: Tree
    atlas: Optional[Atlas]
    mlp: MLP
    queries: Queries
    scene: Optional[Scene] = None
    camera: Optional[Camera] = None
    meta: dict = field(default_factory=dict)


# ------------------------------------------------------------------------------------- generators

def build_tree(scene: Optional[Scene], max_depth: int, uniform: bool = False) -> Tree:
    out = _TreeOut()
    sc = scene._c() if scene is not None else None
    rc = lib().oo_gen_build_tree(C.byref(sc) if sc is not None else None, max_depth, int(uniform), C.byref(out))
    if rc:
        raise RuntimeError("oo_gen_build_tree failed: %d" % rc)
    n = out.n_nodes
    child = np.ctypeslib.as_array(out.child, (n, 8)).copy()
    depth = np.ctypeslib.as_array(out.depth, (n,)).copy()
    coords = np.ctypeslib.as_array(out.coords, (n, 3)).copy()
    for p in (out.child, out.depth, out.coords):
        lib().oo_gen_free(C.cast(p, C.c_void_p))
    depth_first = np.array(out.depth_first[: max_depth + 2], np.int64)
    return Tree(max_depth, child, depth, coords, depth_first)


def make_atlas(tree: Tree, F: int, dtype: str, seed: int, std: float = 0.1, levels=None) -> Atlas:
    """fp16: N(0, std) (A18: std, not variance); fp32 (config 0): U(-1, 1)."""
    out = []
    for l, (R, S) in enumerate(zip(tree.level_res, tree.level_slots)):
        n = S * R * R * F
        if levels is not None and l not in levels:
            out.append(None)
            continue
        if dtype == "f16":
            a = normal_f16(seed, STREAM_ATLAS + l, n, std)
        elif dtype == "f32":
            a = uniform_f32(seed, STREAM_ATLAS + l, n, -1.0, 1.0)
        else:
            raise ValueError(dtype)
        out.append(a.reshape(S, R, R, F))
    return Atlas(F, dtype, out)


def tie_vertex_map_borders(a: np.ndarray) -> np.ndarray:
    """In place: give the boundary vertices of vertex-stored octahedral maps [..][n+1][n+1][F] the values of the vertices
    they coincide with on the sphere ("the edge vertices are shared along adjacent faces", Fig. 3 caption):
    (i, 0) = (n-i, 0), (i, n) = (n-i, n), (0, j) = (0, n-j), (n, j) = (n, n-j); the four corners are all the -z pole.
    Input structure only (which stored entries are one and the same vertex), no interpolation arithmetic."""
    n = a.shape[-2] - 1
    for i in range(n // 2 + 1, n + 1):
        a[..., 0, i, :] = a[..., 0, n - i, :]
        a[..., n, i, :] = a[..., n, n - i, :]
        a[..., i, 0, :] = a[..., n - i, 0, :]
        a[..., i, n, :] = a[..., n - i, n, :]
    a[..., 0, n, :] = a[..., 0, 0, :]
    a[..., n, 0, :] = a[..., 0, 0, :]
    a[..., n, n, :] = a[..., 0, 0, :]
    return a


def make_vertex_atlas(tree: Tree, F: int, dtype: str, seed: int, std: float = 0.1, tie: bool = True) -> Atlas:
    """Vertex-stored maps (PAPER.md "features are stored at map vertices", vertex resolution n_l + 1 with n_l =
    tree.level_res[l] intervals per axis): per used level [slots][n+1][n+1][F], same value distributions as make_atlas,
    boundary vertices tied (tie_vertex_map_borders) unless tie=False (a cache whose owner stored the coinciding vertices
    independently: what the library's upload has to repair)."""
    out = []
    for l, (R, S) in enumerate(zip(tree.level_res, tree.level_slots)):
        n = S * (R + 1) * (R + 1) * F
        a = normal_f16(seed, STREAM_ATLAS + l, n, std) if dtype == "f16" else uniform_f32(seed, STREAM_ATLAS + l, n, -1.0, 1.0)
        a = a.reshape(S, R + 1, R + 1, F)
        out.append(tie_vertex_map_borders(a) if tie else a)
    return Atlas(F, dtype, out)


def disparity(n: int, seed: int, lo: float = 0.25, hi: float = 4.0) -> np.ndarray:
    """Per-query disparity d^ (Eq. 7 output) as a synthetic input: U(lo, hi), i.e. virtual reflected points
    0.25 .. 4 scene units away along the mirror direction."""
    return uniform_f32(seed, STREAM_DISPARITY, n, lo, hi)


def albedo_roughness(n: int, seed: int) -> np.ndarray:
    """[n][4] = diffuse albedo a ~ U(0,1)^3 and roughness alpha ~ U(0.05,1): the extras of PAPER.md Eq. 12."""
    a = uniform_f32(seed, STREAM_ALBEDO, 3 * n, 0.0, 1.0).reshape(n, 3)
    return np.ascontiguousarray(np.concatenate([a, roughness(n, seed)], 1))


def make_mlp(in_dim: int, n_hidden: int, seed: int, width: int = 64, out_dim: int = 3, out_act: str = "exp") -> MLP:
    """He-normal: W ~ N(0, 2/fan_in), no biases, rounded to fp16 (A10, A24)."""
    dims = [in_dim] + [width] * n_hidden + [out_dim]
    ws = []
    for k in range(n_hidden + 1):
        fan_in, fan_out = dims[k], dims[k + 1]
        w = normal(seed, STREAM_WEIGHTS + k, fan_in * fan_out) * np.sqrt(2.0 / fan_in)
        ws.append(f64_to_f16(w).reshape(fan_out, fan_in))
    return MLP(in_dim, width, n_hidden, out_dim, ws, out_act)


@dataclass
class DisparityNet:
    """The disparity predictor g_psi of PAPER.md Eq. 7 as data: a multi-resolution hash grid over position plus a small MLP
    (DESIGN.md §14 lists the hyper-parameters the paper leaves open)."""
    res: List[int]                 # N_g: intervals per axis of level g, coarse -> fine
    hash_log2: int                 # hashed levels have 2^hash_log2 entries; a level with (N_g+1)^3 <= that is dense
    tables: List[np.ndarray]       # fp16 [T_g][Fh]
    weights: List[np.ndarray]      # fp16 [64][G*Fh+3], [64][64], [1][64]

    @property
    def n_features(self) -> int:
        return int(self.tables[0].shape[1])


def hashgrid_resolutions(n_levels: int, n_min: int, n_max: int) -> List[int]:
    """Geometric progression N_g = floor(N_min * b^g), b = (N_max/N_min)^(1/(G-1)) (the schedule of the paper's ref. [25])."""
    if n_levels == 1:
        return [int(n_min)]
    b = np.exp((np.log(n_max) - np.log(n_min)) / (n_levels - 1))
    return [int(np.floor(n_min * b ** g + 1e-9)) for g in range(n_levels)]


def make_disparity_net(seed: int, n_levels: int = 8, n_min: int = 16, n_max: int = 512, hash_log2: int = 17, n_features: int = 2,
                       n_hidden: int = 2, std: float = 0.5, res=None) -> DisparityNet:
    """Seeded stand-in for a trained g_psi: table entries ~ N(0, std) in fp16, weights He-normal fp16, no biases."""
    res = hashgrid_resolutions(n_levels, n_min, n_max) if res is None else [int(r) for r in res]
    tables = []
    for g, N in enumerate(res):
        T = (N + 1) ** 3 if (N + 1) ** 3 <= (1 << hash_log2) else (1 << hash_log2)
        tables.append(normal_f16(seed, STREAM_HASHGRID + g, T * n_features, std).reshape(T, n_features))
    dims = [len(res) * n_features + 3] + [64] * n_hidden + [1]
    ws = []
    for k in range(n_hidden + 1):
        w = normal(seed, STREAM_DISP_WEIGHTS + k, dims[k] * dims[k + 1]) * np.sqrt(2.0 / dims[k])
        ws.append(f64_to_f16(w).reshape(dims[k + 1], dims[k]))
    return DisparityNet(res, hash_log2, tables, ws)


def random_queries(n: int, seed: int, n_extra: int = 0) -> Queries:
    """Config 0: x ~ U[0,1)^3, n uniform on the sphere, wo uniform on the hemisphere about n (A21)."""
    x = uniform_f32(seed, STREAM_POS, 3 * n, 0.0, 1.0).reshape(n, 3)
    nrm = np.empty((n, 3), np.float32)
    wo = np.empty((n, 3), np.float32)
    lib().oo_gen_normals_and_dirs(seed, STREAM_NRM, STREAM_DIR, 0, n, _ptr(nrm), _ptr(wo))
    extra = roughness(n, seed) if n_extra else None
    return Queries(x, nrm, wo, extra)


def roughness(n: int, seed: int) -> np.ndarray:
    return uniform_f32(seed, STREAM_ROUGH, n, 0.05, 1.0).reshape(n, 1)


NOMINAL_EYE = np.array([0.5, 0.5, 0.93])
NOMINAL_LOOK = np.array([0.5, 0.4, 0.3])


def make_scene(kind: str, seed: int) -> Scene:
    """kind "three": 3 spheres r~U(.10,.18) inside the box, no overlap (configs 1, 2);
    kind "many": 64 spheres r~U(.02,.07), centres U[.1,.9]^3, overlap allowed (configs 3, 4).
    Spheres closer than r+0.1 (r+0.05 for "many") to the nominal eye are rejected so that the camera is never
    inside one."""
    lo, hi = 0.03, 0.97
    n_target = 3 if kind == "three" else 64
    u = u01(seed, STREAM_SCENE, 4 * 4096)
    spheres, k = [], 0
    while len(spheres) < n_target:
        a = u[4 * k: 4 * k + 4]
        k += 1
        if kind == "three":
            r = 0.10 + 0.08 * a[3]
            c = (lo + r) + (hi - lo - 2 * r) * a[:3]
            if np.linalg.norm(c - NOMINAL_EYE) < r + 0.1:
                continue
            if any(np.linalg.norm(c - s[:3]) < r + s[3] + 0.01 for s in spheres):
                continue
        else:
            r = 0.02 + 0.05 * a[3]
            c = 0.1 + 0.8 * a[:3]
            if np.linalg.norm(c - NOMINAL_EYE) < r + 0.05:
                continue
        spheres.append(np.array([c[0], c[1], c[2], r]))
    return Scene(np.array(spheres), lo, hi, 1e-5)


def make_camera(width: int, height: int, seed: int) -> Camera:
    j = u01(seed, STREAM_CAMERA, 6) * 0.06 - 0.03
    return Camera(NOMINAL_EYE + j[:3], NOMINAL_LOOK + j[3:], width, height)


def raycast(scene: Scene, cam: Camera, with_surf: bool = False):
    n = cam.width * cam.height
    x = np.empty((n, 3), np.float32)
    nrm = np.empty((n, 3), np.float32)
    wo = np.empty((n, 3), np.float32)
    surf = np.empty(n, np.int32)
    sc, cc = scene._c(), cam._c()
    misses = lib().oo_gen_raycast(C.byref(sc), C.byref(cc), 0, cam.height, _ptr(x), _ptr(nrm), _ptr(wo), _ptr(surf))
    if misses:
        raise RuntimeError("%d primary rays missed the scene" % misses)
    q = Queries(x, nrm, wo)
    return (q, surf) if with_surf else q


def incoherent_queries(scene: Scene, n: int, seed: int, first: int = 0) -> Queries:
    x = np.empty((n, 3), np.float32)
    nrm = np.empty((n, 3), np.float32)
    wo = np.empty((n, 3), np.float32)
    sc = scene._c()
    lib().oo_gen_incoherent(C.byref(sc), seed, STREAM_INCOH, first, n, _ptr(x), _ptr(nrm), _ptr(wo))
    return Queries(x, nrm, wo)


def shuffle_perm(n: int, seed: int) -> np.ndarray:
    """Seeded random permutation (argsort of counter-based uniforms; ties impossible in practice)."""
    return np.argsort(u01(seed, STREAM_SHUFFLE, n), kind="stable").astype(np.uint32)


# ------------------------------------------------------------------------------------------ configs

_LEVELS = {
    1: ([2, 4, 6, 8], [32, 16, 8, 4], 8, 3),             # depths, R_l, F, hidden layers
    3: ([2, 4, 6, 8, 10], [64, 32, 16, 8, 4], 16, 4),
}


def config0(seed: int = 0, n: int = 4096, root0_variant: bool = False) -> Workload:
    """BASELINE.json configs[0]. 73-node uniform tree (1+8+64; "depth 3" counts the root as depth 1, A19),
    used levels = the 8-node and the 64-node level, R = 8, F = 4 fp32 ~ U(-1,1); MLP 14->64->64->3, exp.
    ``root0_variant``: the 585-node tree with used depths {2,3} (the other reading of A19), as an extra test."""
    if root0_variant:
        tree = build_tree(None, 3, uniform=True).set_levels([2, 3], [8, 8])
    else:
        tree = build_tree(None, 2, uniform=True).set_levels([1, 2], [8, 8])
    atlas = make_atlas(tree, 4, "f32", seed)
    mlp = make_mlp(2 * 4 + 6, 2, seed)
    return Workload("cfg0" + ("_root0" if root0_variant else ""), tree, atlas, mlp, random_queries(n, seed))


def scene_workload(cfg: int, seed: int = 0, width: Optional[int] = None, height: Optional[int] = None,
                   with_atlas: bool = True, max_depth: Optional[int] = None, incoherent_n: int = 0,
                   extra_rough: bool = False) -> Workload:
    """configs 1-4. cfg 1: three-sphere scene, depth 8, 1024x1024. cfg 2: same at 1280x720 + roughness.
    cfg 3: 64-sphere scene, depth 10, 2048x2048. ``max_depth`` truncates the level list (reduced-size test
    variants of the same recipe). ``incoherent_n`` > 0 replaces the camera frame by the incoherent sampler (cfg 4)."""
    base = 1 if cfg in (1, 2) else 3
    depths, res, F, H = _LEVELS[base]
    if max_depth is not None:
        keep = [k for k, d in enumerate(depths) if d <= max_depth]
        depths, res = [depths[k] for k in keep], [res[k] for k in keep]
    scene = make_scene("three" if base == 1 else "many", seed)
    if width is None:
        width, height = {1: (1024, 1024), 2: (1280, 720), 3: (2048, 2048), 4: (4096, 4096)}[cfg]
    tree = build_tree(scene, depths[-1]).set_levels(depths, res)
    atlas = make_atlas(tree, F, "f16", seed) if with_atlas else None
    cam = None
    if incoherent_n:
        q = incoherent_queries(scene, incoherent_n, seed)
    else:
        cam = make_camera(width, height, seed)
        q = raycast(scene, cam)
    n_extra = 1 if (cfg == 2 or extra_rough) else 0
    if n_extra:
        q.extra = roughness(q.n, seed)
    mlp = make_mlp(len(depths) * F + 6 + n_extra, H, seed)
    return Workload("cfg%d" % cfg, tree, atlas, mlp, q, scene, cam,
                    {"width": width, "height": height, "n_extra": n_extra})


def paper_workload(seed: int = 0, width: int = 1024, height: int = 1024, depths=None, res=None, F: int = 4,
                   dtype: str = "f32", width_mlp: int = 128, n_hidden: int = 4, incoherent_n: int = 0) -> Workload:
    """The paper's own shapes (PAPER.md "Implementation details": K = 8 consecutive levels with spatial resolution
    (2^2)^3 .. (2^9)^3, vertex resolution 2^8+1 .. 2^1+1, C = 4 features per vertex; decoder 4 hidden layers x 128) on the
    three-sphere stand-in scene of config 1: used depths 2..9, R_l = 256 .. 2 intervals (vertex maps, fp32 as Table 2's
    16 bytes per entry implies), queries = the primary hits of a width x height frame plus the attributes of Eq. 12
    (albedo, roughness as extras) and a synthetic per-query disparity (Eq. 7's output).  ``depths``/``res`` give reduced
    variants of the same recipe for tests.  meta["disparity"] holds d^, meta["dirmap"] = "vertex"."""
    depths = list(range(2, 10)) if depths is None else [int(d) for d in depths]
    res = [1 << (10 - d) for d in depths] if res is None else [int(r) for r in res]
    scene = make_scene("three", seed)
    tree = build_tree(scene, depths[-1]).set_levels(depths, res)
    atlas = make_vertex_atlas(tree, F, dtype, seed)
    cam = None
    if incoherent_n:
        q = incoherent_queries(scene, incoherent_n, seed)
    else:
        cam = make_camera(width, height, seed)
        q = raycast(scene, cam)
    q.extra = albedo_roughness(q.n, seed)
    mlp = make_mlp(len(depths) * F + 9 + 4, n_hidden, seed, width=width_mlp)
    return Workload("paper", tree, atlas, mlp, q, scene, cam,
                    {"width": width, "height": height, "n_extra": 4, "disparity": disparity(q.n, seed), "dirmap": "vertex"})
