"""ctypes binding of oracle/oo_oracle.c (the plain-C double-precision oracle). TEST INFRASTRUCTURE ONLY."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oo_oracle.c")
_LIB = os.path.join(_HERE, "liboo_oracle.so")
MAX_LEVELS, MAX_LAYERS = 16, 16


def build_lib(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Tree(C.Structure):
    _fields_ = [("n_nodes", C.c_uint32), ("max_depth", C.c_uint32), ("child", C.c_void_p), ("map_slot", C.c_void_p),
                ("n_levels", C.c_uint32), ("level_depth", C.c_uint32 * MAX_LEVELS), ("level_res", C.c_uint32 * MAX_LEVELS),
                ("n_features", C.c_uint32), ("dtype", C.c_int32), ("atlas", C.c_void_p * MAX_LEVELS)]


class _Mlp(C.Structure):
    _fields_ = [("in_dim", C.c_uint32), ("width", C.c_uint32), ("n_hidden", C.c_uint32), ("out_dim", C.c_uint32),
                ("weights", C.c_void_p * MAX_LAYERS), ("out_act", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build_lib())
        L.oracle_max_threads.restype = C.c_int
        L.oracle_encode.restype = C.c_int
        L.oracle_encode.argtypes = [C.POINTER(_Tree), C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_void_p, C.c_int]
        L.oracle_query.restype = C.c_int
        L.oracle_query.argtypes = [C.POINTER(_Tree), C.POINTER(_Mlp), C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p,
                                   C.c_void_p, C.c_uint32, C.c_void_p, C.c_int]
        _lib = L
    return _lib


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def _f32(a):
    a = np.ascontiguousarray(a, np.float32)
    return a


class COracle:
    """Holds references to the host arrays (tree, atlas, weights) for the lifetime of the object."""

    def __init__(self, tree, atlas_levels, atlas_dtype: str, mlp_weights=None, out_act: str = "exp"):
        self._keep = []
        child = np.ascontiguousarray(tree.child, np.int32)
        slot = np.ascontiguousarray(tree.map_slot, np.int32)
        self._keep += [child, slot]
        t = _Tree()
        t.n_nodes, t.max_depth = child.shape[0], tree.max_depth
        t.child, t.map_slot = child.ctypes.data, slot.ctypes.data
        t.n_levels = len(tree.level_depth)
        want = np.float16 if atlas_dtype == "f16" else np.float32
        for l, (d, R) in enumerate(zip(tree.level_depth, tree.level_res)):
            t.level_depth[l], t.level_res[l] = d, R
            a = np.ascontiguousarray(atlas_levels[l], want)
            assert a.shape[1] == R and a.shape[2] == R
            self._keep.append(a)
            t.atlas[l] = a.ctypes.data
            t.n_features = a.shape[3]
        t.dtype = 0 if atlas_dtype == "f16" else 1
        self.tree, self.L, self.F = t, int(t.n_levels), int(t.n_features)
        self.mlp = None
        if mlp_weights is not None:
            m = _Mlp()
            m.in_dim, m.width = mlp_weights[0].shape[1], mlp_weights[0].shape[0]
            m.n_hidden, m.out_dim = len(mlp_weights) - 1, mlp_weights[-1].shape[0]
            for k, w in enumerate(mlp_weights):
                w = np.ascontiguousarray(w, np.float16)
                self._keep.append(w)
                m.weights[k] = w.ctypes.data
            m.out_act = {"none": 0, "exp": 1}[out_act]
            self.mlp = m

    def encode(self, x, wo, n_threads: int = 0):
        x, wo = _f32(x), _f32(wo)
        n = x.shape[0]
        feat = np.empty((n, self.L * self.F), np.float64)
        slot = np.empty((n, self.L), np.int32)
        tex = np.empty((n, self.L, 2), np.int16)
        rc = lib().oracle_encode(C.byref(self.tree), n, x.ctypes.data, wo.ctypes.data, feat.ctypes.data,
                                 slot.ctypes.data, tex.ctypes.data, n_threads)
        if rc < 0:
            raise RuntimeError("oracle_encode: %d" % rc)
        return feat, slot, tex

    def query(self, x, nrm, wo, extra=None, n_threads: int = 0, return_threads: bool = False):
        assert self.mlp is not None
        x, nrm, wo = _f32(x), _f32(nrm), _f32(wo)
        n = x.shape[0]
        n_extra = 0
        ep = None
        if extra is not None:
            extra = _f32(extra).reshape(n, -1)
            n_extra, ep = extra.shape[1], extra.ctypes.data
        rgb = np.empty((n, int(self.mlp.out_dim)), np.float64)
        rc = lib().oracle_query(C.byref(self.tree), C.byref(self.mlp), n, x.ctypes.data, nrm.ctypes.data,
                                wo.ctypes.data, ep, n_extra, rgb.ctypes.data, n_threads)
        if rc < 0:
            raise RuntimeError("oracle_query: %d" % rc)
        return (rgb, rc) if return_threads else rgb


def from_workload(w, with_mlp: bool = True) -> COracle:
    return COracle(w.tree, w.atlas.levels, w.atlas.dtype, w.mlp.weights if with_mlp else None, w.mlp.out_act)
