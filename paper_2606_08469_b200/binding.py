"""ctypes binding of liboo (include/oo.h): same names, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboo.so")

PATH_AUTO, PATH_GENERIC, PATH_UNFUSED, PATH_FUSED_MMA, PATH_FUSED_TC, PATH_FUSED_TC_TMEM, PATH_FULL = 0, 1, 2, 3, 4, 5, 6
SPATIAL = {"nearest": 0, "trilinear8": 1}
DIRMAP = {"texel": 0, "vertex": 1}
LOOKUP = {"wo": 0, "mirror": 1, "shifted": 2}
ATTRS = {"n_wo": 0, "paper": 1}
OO_F16, OO_F32 = 0, 1
OO_ACT_NONE, OO_ACT_EXP = 0, 1
_STATUS = {0: "OO_OK", 1: "OO_ERR_INVALID_ARG", 2: "OO_ERR_NOT_READY", 3: "OO_ERR_UNSUPPORTED", 4: "OO_ERR_CUDA", 5: "OO_ERR_OOM"}

EXPORTED_SYMBOLS = ["oo_create", "oo_destroy", "oo_last_error", "oo_upload_tree", "oo_upload_mlp", "oo_reserve", "oo_set_path",
                    "oo_get_info", "oo_sort_queries", "oo_encode", "oo_query", "oo_query_host", "oo_read_padded_map", "oo_set_mode",
                    "oo_encode_full", "oo_upload_scene", "oo_raycast", "oo_upload_disparity", "oo_predict_disparity", "oo_set_presort",
                    "oo_query_debug", "oo_set_host_chunks", "oo_last_note", "oo_set_host_zero_copy", "oo_sort_queries_static"]


class OOError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__("%s: %s" % (_STATUS.get(status, str(status)), msg))
        self.status = status


class _TreeDesc(C.Structure):
    _fields_ = [("n_nodes", C.c_uint32), ("max_depth", C.c_uint32), ("child", C.c_void_p), ("depth", C.c_void_p),
                ("map_slot", C.c_void_p), ("n_levels", C.c_uint32), ("level_depth", C.c_void_p), ("level_res", C.c_void_p),
                ("level_slots", C.c_void_p), ("n_features", C.c_uint32), ("dtype", C.c_int), ("atlas", C.c_void_p),
                ("dirmap", C.c_int)]


class _MlpDesc(C.Structure):
    _fields_ = [("in_dim", C.c_uint32), ("width", C.c_uint32), ("n_hidden", C.c_uint32), ("out_dim", C.c_uint32),
                ("weights", C.c_void_p), ("out_act", C.c_int), ("weights_on_device", C.c_uint32)]


class _Queries(C.Structure):
    _fields_ = [("n", C.c_uint64), ("x", C.c_void_p), ("nrm", C.c_void_p), ("wo", C.c_void_p), ("extra", C.c_void_p),
                ("n_extra", C.c_uint32), ("perm", C.c_void_p), ("disparity", C.c_void_p)]


class _DisparityDesc(C.Structure):
    _fields_ = [("n_levels", C.c_uint32), ("n_features", C.c_uint32), ("res", C.c_void_p), ("hash_log2", C.c_uint32),
                ("tables", C.c_void_p), ("n_hidden", C.c_uint32), ("weights", C.c_void_p)]


class _SceneDesc(C.Structure):
    _fields_ = [("n_spheres", C.c_uint32), ("spheres", C.c_void_p), ("lo", C.c_double), ("hi", C.c_double)]


class _CameraDesc(C.Structure):
    _fields_ = [("eye", C.c_double * 3), ("look", C.c_double * 3), ("up", C.c_double * 3), ("vfov_deg", C.c_double),
                ("width", C.c_uint32), ("height", C.c_uint32)]


class _Mode(C.Structure):
    _fields_ = [("spatial", C.c_int), ("lookup", C.c_int), ("attrs", C.c_int)]


class _Info(C.Structure):
    _fields_ = [("launches", C.c_uint64), ("query_launches", C.c_uint64), ("node_table_bytes", C.c_uint64),
                ("atlas_bytes", C.c_uint64), ("path_last_query", C.c_uint32), ("path_last_encode", C.c_uint32),
                ("hop_plan_ok", C.c_uint32), ("n_sms", C.c_uint32),
                ("presorted_last_query", C.c_uint32), ("presorted_last_encode", C.c_uint32),
                ("full_query", C.c_uint32), ("n_neighbours", C.c_uint32), ("tied_vertices", C.c_uint64), ("host_zero_copy_last", C.c_uint32), ("presort_auto_on", C.c_uint32),
                ("coherence_x100", C.c_uint32), ("encode_pipelined_last", C.c_uint32)]


_lib = None


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """Load liboo.so.  Fails loudly if it has not been built (python -m paper_2606_08469_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise OOError(4, "liboo.so is not built (%s); run `python -m paper_2606_08469_b200.build` — there is no CPU fallback" % _LIB_PATH)
    L = C.CDLL(_LIB_PATH)
    vp, u64, u32 = C.c_void_p, C.c_uint64, C.c_uint32
    L.oo_create.argtypes = [C.POINTER(vp), C.c_int]
    L.oo_destroy.argtypes = [vp]
    L.oo_destroy.restype = None
    L.oo_last_error.argtypes = [vp]
    L.oo_last_error.restype = C.c_char_p
    L.oo_last_note.argtypes = [vp]
    L.oo_last_note.restype = C.c_char_p
    L.oo_query_debug.argtypes = [vp, C.POINTER(_Queries), vp, vp, vp, vp]
    L.oo_set_host_chunks.argtypes = [vp, u32]
    L.oo_set_host_zero_copy.argtypes = [vp, u32]
    L.oo_upload_tree.argtypes = [vp, C.POINTER(_TreeDesc), vp]
    L.oo_upload_mlp.argtypes = [vp, C.POINTER(_MlpDesc), vp]
    L.oo_reserve.argtypes = [vp, u64]
    L.oo_set_path.argtypes = [vp, C.c_int]
    L.oo_get_info.argtypes = [vp, C.POINTER(_Info)]
    L.oo_set_presort.argtypes = [vp, C.c_int, u64]
    L.oo_sort_queries.argtypes = [vp, C.POINTER(_Queries), vp, vp]
    L.oo_sort_queries_static.argtypes = [vp, u64, vp, vp, C.c_char_p, C.c_size_t]
    L.oo_encode.argtypes = [vp, C.POINTER(_Queries), vp, vp, vp, vp]
    L.oo_query.argtypes = [vp, C.POINTER(_Queries), vp, vp]
    L.oo_query_host.argtypes = [vp, C.POINTER(_Queries), vp, vp]
    L.oo_read_padded_map.argtypes = [vp, u32, u32, vp]
    L.oo_set_mode.argtypes = [vp, C.POINTER(_Mode)]
    L.oo_upload_scene.argtypes = [vp, C.POINTER(_SceneDesc), vp]
    L.oo_raycast.argtypes = [vp, C.POINTER(_CameraDesc), vp, vp, vp, vp, vp]
    L.oo_encode_full.argtypes = [vp, C.POINTER(_Queries), vp, vp, vp, vp]
    L.oo_upload_disparity.argtypes = [vp, C.POINTER(_DisparityDesc), vp]
    L.oo_predict_disparity.argtypes = [vp, C.POINTER(_Queries), vp, vp, vp]
    for name in EXPORTED_SYMBOLS:
        if name not in ("oo_destroy", "oo_last_error", "oo_last_note"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p)


SORT_STATIC_MAX_QUERIES = 1 << 20      # OO_SORT_STATIC_MAX_QUERIES


def oo_sort_queries_static(x, perm_out=None):
    """Morton order of the positions `x` (CUDA fp32 tensor [n][3]) without any device allocation inside the library: the variant
    of `OctaOctree.oo_sort_queries` for callers that cannot allocate (fixed memory budget after start-up, a host application that
    owns the device heap, a latency-critical thread).  Needs no context and no oo_reserve; at most SORT_STATIC_MAX_QUERIES
    positions, more raises OOError(OO_ERR_UNSUPPORTED).  Runs on x's device and on torch's current stream for it.  Pass
    `perm_out` (int32/uint32 CUDA tensor [n]) to keep this wrapper from allocating the result as well.  Calls share one
    built-in scratch array per device: do not let two of them overlap on the GPU (see include/oo.h)."""
    import torch  # device memory and streams only
    L = load_library()
    assert x.is_cuda and x.is_contiguous() and x.dtype == torch.float32, "x must be a contiguous fp32 CUDA tensor"
    n = int(x.shape[0])
    if perm_out is None:
        perm_out = torch.empty(n, dtype=torch.int32, device=x.device)
    assert perm_out.is_cuda and perm_out.is_contiguous() and perm_out.element_size() == 4 and perm_out.numel() >= n
    err = C.create_string_buffer(256)
    with torch.cuda.device(x.device):      # the entry point works on the calling thread's current device
        st = L.oo_sort_queries_static(C.c_void_p(x.data_ptr()), n, C.c_void_p(perm_out.data_ptr()),
                                      C.c_void_p(torch.cuda.current_stream(x.device).cuda_stream), err, len(err))
    if st:
        raise OOError(st, err.value.decode())
    return perm_out


class OctaOctree:
    """One context on one CUDA device.  Methods mirror the C entry points (oo_upload_tree, oo_upload_mlp, oo_encode,
    oo_query, oo_sort_queries, oo_query_host); tensors are torch CUDA tensors, trees/weights are numpy arrays."""

    def __init__(self, device: int = 0):
        import torch  # device memory and streams only
        self._torch = torch
        self._L = load_library()
        self._ctx = C.c_void_p()
        st = self._L.oo_create(C.byref(self._ctx), device)
        if st:
            raise OOError(st, "oo_create(device=%d) failed: needs a CUDA device of compute capability 10.x (B200); there is no CPU fallback" % device)
        self.device = torch.device("cuda", device)
        self.n_levels = self.n_features = 0
        self.dtype = None
        self.out_dim = 3
        self.n_neighbours = 1

    def close(self):
        if self._ctx:
            self._L.oo_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st:
            raise OOError(st, self._L.oo_last_error(self._ctx).decode())

    def _stream(self):
        return C.c_void_p(self._torch.cuda.current_stream(self.device).cuda_stream)

    # ---------------------------------------------------------------- uploads
    def oo_upload_tree(self, tree, atlas_levels: Sequence, dtype: str, dirmap: str = "texel"):
        """tree: object with n_nodes, max_depth, child, depth, map_slot, level_depth, level_res, level_slots (numpy / lists).
        atlas_levels: per level a numpy array or a torch CUDA tensor [slots][R][R][F] (dirmap "vertex": [slots][R+1][R+1][F])."""
        import numpy as np
        torch = self._torch
        child = np.ascontiguousarray(tree.child, np.int32)
        depth = np.ascontiguousarray(tree.depth, np.uint8)
        slot = np.ascontiguousarray(tree.map_slot, np.int32)
        ld = np.ascontiguousarray(tree.level_depth, np.uint32)
        lr = np.ascontiguousarray(tree.level_res, np.uint32)
        ls = np.ascontiguousarray(tree.level_slots, np.uint32)
        tdt = {"f16": torch.float16, "f32": torch.float32}[dtype]
        dev = []
        for a in atlas_levels:
            t = a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a))
            t = t.to(device=self.device, dtype=tdt).contiguous()
            dev.append(t)
        F = int(dev[0].shape[-1])
        ptrs = (C.c_void_p * len(dev))(*[t.data_ptr() if t.numel() else None for t in dev])
        d = _TreeDesc(child.shape[0], int(tree.max_depth), _np_ptr(child), _np_ptr(depth), _np_ptr(slot), len(dev), _np_ptr(ld),
                      _np_ptr(lr), _np_ptr(ls), F, OO_F16 if dtype == "f16" else OO_F32, C.cast(ptrs, C.c_void_p), DIRMAP[dirmap])
        self._check(self._L.oo_upload_tree(self._ctx, C.byref(d), self._stream()))
        self.n_levels, self.n_features, self.dtype = len(dev), F, dtype
        del dev

    def oo_upload_mlp(self, weights: Sequence, out_act: str = "exp"):
        """weights: fp16 matrices [out][in], numpy arrays (host) or torch CUDA tensors (oo_mlp_desc.weights_on_device)."""
        import numpy as np
        torch = self._torch
        on_dev = all(isinstance(w, torch.Tensor) and w.is_cuda for w in weights)
        if on_dev:
            ws = [w.to(dtype=torch.float16).contiguous() for w in weights]
            ptrs = (C.c_void_p * len(ws))(*[w.data_ptr() for w in ws])
        else:
            ws = [np.ascontiguousarray(w, np.float16) for w in weights]
            ptrs = (C.c_void_p * len(ws))(*[w.ctypes.data for w in ws])
        d = _MlpDesc(ws[0].shape[1], ws[0].shape[0], len(ws) - 1, ws[-1].shape[0], C.cast(ptrs, C.c_void_p),
                     {"none": OO_ACT_NONE, "exp": OO_ACT_EXP}[out_act], 1 if on_dev else 0)
        self._check(self._L.oo_upload_mlp(self._ctx, C.byref(d), self._stream()))
        self.out_dim = int(ws[-1].shape[0])

    def oo_upload_disparity(self, res: Sequence[int], hash_log2: int, tables: Sequence, weights: Sequence):
        """The disparity predictor g_psi (Eq. 7): per-level resolutions, fp16 tables [T_g][2], fp16 weights."""
        import numpy as np
        r = np.ascontiguousarray(res, np.uint32)
        ts = [np.ascontiguousarray(t, np.float16) for t in tables]
        ws = [np.ascontiguousarray(w, np.float16) for w in weights]
        tp = (C.c_void_p * len(ts))(*[t.ctypes.data for t in ts])
        wp = (C.c_void_p * len(ws))(*[w.ctypes.data for w in ws])
        d = _DisparityDesc(len(ts), int(ts[0].shape[1]), _np_ptr(r), int(hash_log2), C.cast(tp, C.c_void_p), len(ws) - 1, C.cast(wp, C.c_void_p))
        self._check(self._L.oo_upload_disparity(self._ctx, C.byref(d), self._stream()))
        self.n_grid_levels = len(ts)

    def oo_predict_disparity(self, x, nrm, wo, want_features: bool = False, disparity=None):
        """d^ [n] fp32 on the device (and, with want_features, the hash-grid features [n][2G] fp32)."""
        torch = self._torch
        q, n = self._queries(x, nrm, wo, None, None, None)
        if disparity is None:
            disparity = torch.empty(n, dtype=torch.float32, device=self.device)
        feats = torch.empty((n, 2 * self.n_grid_levels), dtype=torch.float32, device=self.device) if want_features else None
        self._check(self._L.oo_predict_disparity(self._ctx, C.byref(q), C.c_void_p(disparity.data_ptr()),
                                                 C.c_void_p(feats.data_ptr()) if want_features else None, self._stream()))
        return (disparity, feats) if want_features else disparity

    def oo_reserve(self, n: int):
        self._check(self._L.oo_reserve(self._ctx, int(n)))

    def oo_set_path(self, path: int):
        self._check(self._L.oo_set_path(self._ctx, int(path)))

    def oo_set_presort(self, presort: str = "auto", min_queries: int = 0):
        """"auto" (the library's default: decided from the coherence of the recent calls), "none", or "bin" (oo_query / oo_encode
        bin the queries by their top Morton bits first; see oo_presort).
        Batches below min_queries proceed unsorted (0 = library default)."""
        self._check(self._L.oo_set_presort(self._ctx, {"none": 0, "bin": 1, "auto": 2}[presort], int(min_queries)))

    def oo_set_mode(self, spatial: str = "nearest", lookup: str = "wo", attrs: str = "n_wo"):
        m = _Mode(SPATIAL[spatial], LOOKUP[lookup], ATTRS[attrs])
        self._check(self._L.oo_set_mode(self._ctx, C.byref(m)))
        self.n_neighbours = 8 if spatial == "trilinear8" else 1

    def oo_get_info(self) -> dict:
        info = _Info()
        self._check(self._L.oo_get_info(self._ctx, C.byref(info)))
        return {k: int(getattr(info, k)) for k, _ in _Info._fields_}

    # ---------------------------------------------------------------- queries
    def _queries(self, x, nrm, wo, extra, perm, disparity=None):
        torch = self._torch
        for t in (x, nrm, wo, extra, perm, disparity):
            if t is not None:
                assert t.is_cuda and t.is_contiguous(), "queries must be contiguous CUDA tensors"
        assert x.dtype == torch.float32 and wo.dtype == torch.float32
        n = int(x.shape[0])
        ne = 0 if extra is None else int(extra.numel() // max(n, 1))
        q = _Queries(n, x.data_ptr(), nrm.data_ptr() if nrm is not None else None, wo.data_ptr(),
                     extra.data_ptr() if extra is not None else None, ne, perm.data_ptr() if perm is not None else None,
                     disparity.data_ptr() if disparity is not None else None)
        return q, n

    def oo_sort_queries(self, x, perm_out=None):
        torch = self._torch
        n = int(x.shape[0])
        if perm_out is None:
            perm_out = torch.empty(n, dtype=torch.int32, device=self.device)
        q = _Queries(n, x.data_ptr(), None, x.data_ptr(), None, 0, None)
        self._check(self._L.oo_sort_queries(self._ctx, C.byref(q), C.c_void_p(perm_out.data_ptr()), self._stream()))
        return perm_out

    def oo_encode(self, x, wo, perm=None, features=None, want_debug: bool = False):
        torch = self._torch
        q, n = self._queries(x, None, wo, None, perm)
        LF = self.n_levels * self.n_features
        if features is None:
            features = torch.empty((n, LF), dtype=torch.float16 if self.dtype == "f16" else torch.float32, device=self.device)
        slot = texel = None
        if want_debug:
            slot = torch.empty((n, self.n_levels), dtype=torch.int32, device=self.device)
            texel = torch.empty((n, self.n_levels, 2), dtype=torch.int16, device=self.device)
        self._check(self._L.oo_encode(self._ctx, C.byref(q), C.c_void_p(features.data_ptr()),
                                      C.c_void_p(slot.data_ptr()) if want_debug else None,
                                      C.c_void_p(texel.data_ptr()) if want_debug else None, self._stream()))
        return (features, slot, texel) if want_debug else features

    def oo_encode_full(self, x, nrm, wo, disparity=None, perm=None, want_debug: bool = False):
        """features fp32 [n][L*F] under the current mode; with want_debug also slots [n][L][J] and cells [n][L][J][3]."""
        torch = self._torch
        q, n = self._queries(x, nrm, wo, None, perm, disparity)
        features = torch.empty((n, self.n_levels * self.n_features), dtype=torch.float32, device=self.device)
        slot = cell = None
        if want_debug:
            slot = torch.empty((n, self.n_levels, self.n_neighbours), dtype=torch.int32, device=self.device)
            cell = torch.empty((n, self.n_levels, self.n_neighbours, 3), dtype=torch.int16, device=self.device)
        self._check(self._L.oo_encode_full(self._ctx, C.byref(q), C.c_void_p(features.data_ptr()),
                                           C.c_void_p(slot.data_ptr()) if want_debug else None,
                                           C.c_void_p(cell.data_ptr()) if want_debug else None, self._stream()))
        return (features, slot, cell) if want_debug else features

    def oo_query(self, x, nrm, wo, extra=None, perm=None, rgb=None, disparity=None):
        torch = self._torch
        q, n = self._queries(x, nrm, wo, extra, perm, disparity)
        if rgb is None:
            rgb = torch.empty((n, self.out_dim), dtype=torch.float32, device=self.device)
        self._check(self._L.oo_query(self._ctx, C.byref(q), C.c_void_p(rgb.data_ptr()), self._stream()))
        return rgb

    def oo_query_debug(self, x, nrm, wo, extra=None, perm=None, rgb=None, disparity=None):
        """oo_query through the fused kernels' debug instances: (rgb, slot, index).  Hot path: slot [n][L] int32, index
        [n][L][2] int16; full query: slot [n][L][J], index [n][L][J][3]."""
        torch = self._torch
        q, n = self._queries(x, nrm, wo, extra, perm, disparity)
        if rgb is None:
            rgb = torch.empty((n, self.out_dim), dtype=torch.float32, device=self.device)
        info = self.oo_get_info()
        full = bool(info["full_query"])
        shape = (n, self.n_levels, info["n_neighbours"]) if full else (n, self.n_levels)
        slot = torch.full(shape, -2, dtype=torch.int32, device=self.device)
        index = torch.full(shape + ((3,) if full else (2,)), -32768, dtype=torch.int16, device=self.device)
        self._check(self._L.oo_query_debug(self._ctx, C.byref(q), C.c_void_p(rgb.data_ptr()), C.c_void_p(slot.data_ptr()),
                                           C.c_void_p(index.data_ptr()), self._stream()))
        return rgb, slot, index

    def oo_set_host_chunks(self, n_chunks: int = 0):
        self._check(self._L.oo_set_host_chunks(self._ctx, int(n_chunks)))

    def oo_set_host_zero_copy(self, enable: bool = True):
        self._check(self._L.oo_set_host_zero_copy(self._ctx, 1 if enable else 0))

    def oo_last_note(self) -> str:
        return self._L.oo_last_note(self._ctx).decode()

    def oo_query_host(self, x, nrm, wo, extra=None, rgb=None, disparity=None):
        """x, nrm, wo, extra, rgb: CPU tensors (pinned for asynchronous copies) or numpy arrays.  Synchronous."""
        torch = self._torch
        n = int(x.shape[0])

        def ptr(a):
            if a is None:
                return None
            return a.data_ptr() if isinstance(a, torch.Tensor) else a.ctypes.data
        ne = 0 if extra is None else int((extra.numel() if isinstance(extra, torch.Tensor) else extra.size) // max(n, 1))
        if rgb is None:
            rgb = torch.empty((n, self.out_dim), dtype=torch.float32).pin_memory()
        q = _Queries(n, ptr(x), ptr(nrm), ptr(wo), ptr(extra), ne, None, ptr(disparity))
        self._check(self._L.oo_query_host(self._ctx, C.byref(q), C.c_void_p(ptr(rgb)), self._stream()))
        return rgb

    def oo_upload_scene(self, spheres, lo: float, hi: float):
        """spheres: [n][4] (centre, radius), float64."""
        import numpy as np
        sp = np.ascontiguousarray(spheres, np.float64).reshape(-1, 4)
        d = _SceneDesc(sp.shape[0], _np_ptr(sp) if sp.shape[0] else None, float(lo), float(hi))
        self._check(self._L.oo_upload_scene(self._ctx, C.byref(d), self._stream()))

    def oo_raycast(self, eye, look, up, vfov_deg: float, width: int, height: int, want_surf: bool = False, out=None):
        """Primary hits of a frame as query tensors (x, nrm, wo[, surf]) on the device, scanline order."""
        torch = self._torch
        n = int(width) * int(height)
        if out is None:
            out = tuple(torch.empty((n, 3), dtype=torch.float32, device=self.device) for _ in range(3))
        x, nrm, wo = out
        surf = torch.empty(n, dtype=torch.int32, device=self.device) if want_surf else None
        cam = _CameraDesc((C.c_double * 3)(*[float(v) for v in eye]), (C.c_double * 3)(*[float(v) for v in look]),
                          (C.c_double * 3)(*[float(v) for v in up]), float(vfov_deg), int(width), int(height))
        self._check(self._L.oo_raycast(self._ctx, C.byref(cam), C.c_void_p(x.data_ptr()), C.c_void_p(nrm.data_ptr()),
                                       C.c_void_p(wo.data_ptr()), C.c_void_p(surf.data_ptr()) if want_surf else None, self._stream()))
        return (x, nrm, wo, surf) if want_surf else (x, nrm, wo)

    def oo_read_padded_map(self, level: int, slot: int, R: int):
        import numpy as np
        out = np.empty((R + 2, R + 2, self.n_features), np.float16 if self.dtype == "f16" else np.float32)
        self._check(self._L.oo_read_padded_map(self._ctx, level, slot, _np_ptr(out)))
        return out

    # convenience: upload a gen.Workload
    def upload_workload(self, w, dirmap: str = "texel"):
        self.oo_upload_tree(w.tree, w.atlas.levels, w.atlas.dtype, dirmap)
        self.oo_upload_mlp(w.mlp.weights, w.mlp.out_act)
        return self
