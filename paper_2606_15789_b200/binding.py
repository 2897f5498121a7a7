"""Thin ctypes binding of libanslin.so (include/anslin.h): argument marshalling only.

Every step of the hot path runs inside the library's kernels; torch is used by CALLERS for device
memory and streams.  There is no fallback: if the shared object is missing or a call fails, an
exception is raised.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libanslin.so")

FMT_BF16, FMT_FP8_E4M3, FMT_INT8, FMT_INT4_AWQ, FMT_FP8_E5M2, FMT_FP4_E2M1, FMT_BF16_PAIR4 = 0, 1, 2, 3, 4, 5, 6
DT_F32, DT_F16, DT_BF16, DT_I8, DT_FP8_E4M3, DT_FP8_E5M2 = 0, 1, 2, 3, 4, 5
FLAG_STATE_PAYLOAD = 1
FLAG_LANE_STREAMS = 2
X_DTYPE = {FMT_BF16: DT_BF16, FMT_FP8_E4M3: DT_FP8_E4M3, FMT_INT8: DT_I8, FMT_INT4_AWQ: DT_F16, FMT_FP8_E5M2: DT_FP8_E5M2, FMT_FP4_E2M1: DT_FP8_E4M3, FMT_BF16_PAIR4: DT_BF16}

EXPORTS = ["anslin_encode_bound", "anslin_encode_host", "anslin_open", "anslin_close", "anslin_describe",
           "anslin_decode", "anslin_gemm_workspace_bytes", "anslin_gemm_multi_workspace_bytes", "anslin_gemm",
           "anslin_gemm_multi", "anslin_gemm_multi_ex", "anslin_gemm_grouped",
           "anslin_dense_workspace_bytes", "anslin_dense_gemm", "anslin_histogram", "anslin_entropy_bits",
           "anslin_entropy_weighted", "anslin_encode_device_workspace_bytes", "anslin_encode_device_head_bytes",
           "anslin_encode_device", "anslin_gemm_launches", "anslin_status_string", "anslin_gemm_static"]


class AnslinError(RuntimeError):
    pass


class Desc(ctypes.Structure):
    _fields_ = [("format", ctypes.c_uint32), ("n_out", ctypes.c_uint32), ("k_in", ctypes.c_uint32),
                ("tile_k", ctypes.c_uint32), ("group_size", ctypes.c_uint32), ("flags", ctypes.c_uint32),
                ("w_scale", ctypes.c_float), ("tile_n", ctypes.c_uint32)]


class Stats(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint64) for n in ("n_weights", "payload_bits", "state_bits", "pad_bits", "offset_table_bits",
                                               "freq_table_bits", "raw_bits", "side_bits", "total_bytes")] + \
               [(n, ctypes.c_double) for n in ("entropy_bits_per_symbol", "xent_bits_per_symbol",
                                               "raw_entropy_bits_per_symbol", "bits_per_weight")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise AnslinError("libanslin.so is not built (run `python -m paper_2606_15789_b200.build`); there is no fallback")
        L = ctypes.CDLL(LIB_PATH)
        vp, sz, i32, u32, i64 = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int32, ctypes.c_uint32, ctypes.c_int64
        L.anslin_encode_bound.argtypes = [ctypes.POINTER(Desc)]; L.anslin_encode_bound.restype = sz
        L.anslin_encode_host.argtypes = [ctypes.POINTER(Desc), vp, vp, vp, vp, sz, ctypes.POINTER(sz), ctypes.POINTER(Stats)]
        L.anslin_open.argtypes = [vp, sz, vp, ctypes.POINTER(vp)]
        L.anslin_close.argtypes = [vp]
        L.anslin_describe.argtypes = [vp, ctypes.POINTER(Desc)]
        L.anslin_decode.argtypes = [vp, vp, sz, vp]
        L.anslin_gemm_workspace_bytes.argtypes = [vp, i32]; L.anslin_gemm_workspace_bytes.restype = sz
        L.anslin_gemm.argtypes = [vp, vp, u32, i64, i32, vp, vp, i64, vp, sz, vp]
        L.anslin_gemm_static.argtypes = [vp, vp, u32, i64, i32, vp, vp, i64, vp]
        L.anslin_gemm_multi_workspace_bytes.argtypes = [ctypes.POINTER(vp), i32, i32]
        L.anslin_gemm_multi_workspace_bytes.restype = sz
        L.anslin_gemm_multi.argtypes = [ctypes.POINTER(vp), i32, ctypes.POINTER(vp), u32, ctypes.POINTER(i64), ctypes.POINTER(i32),
                                        ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i64), vp, sz, vp]
        L.anslin_gemm_multi_ex.argtypes = [ctypes.POINTER(vp), i32, ctypes.POINTER(vp), u32, ctypes.POINTER(i64), ctypes.POINTER(i32),
                                           ctypes.POINTER(vp), ctypes.POINTER(vp), u32, ctypes.POINTER(i64), vp, sz, vp]
        L.anslin_gemm_grouped.argtypes = [ctypes.POINTER(vp), i32, ctypes.POINTER(i32), vp, u32, i64, vp, vp, i64, vp, sz, vp]
        L.anslin_dense_workspace_bytes.argtypes = [u32, u32, i32]; L.anslin_dense_workspace_bytes.restype = sz
        L.anslin_dense_gemm.argtypes = [u32, vp, u32, u32, vp, ctypes.c_float, vp, u32, i64, i32, vp, vp, i64, vp, sz, vp]
        L.anslin_histogram.argtypes = [u32, vp, ctypes.c_uint64, vp, vp]
        L.anslin_entropy_bits.argtypes = [ctypes.POINTER(ctypes.c_uint64), i32]; L.anslin_entropy_bits.restype = ctypes.c_double
        L.anslin_entropy_weighted.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_uint64), i32]
        L.anslin_entropy_weighted.restype = ctypes.c_double
        L.anslin_encode_device_workspace_bytes.argtypes = [ctypes.POINTER(Desc)]; L.anslin_encode_device_workspace_bytes.restype = sz
        L.anslin_encode_device_head_bytes.argtypes = [ctypes.POINTER(Desc)]; L.anslin_encode_device_head_bytes.restype = sz
        L.anslin_encode_device.argtypes = [ctypes.POINTER(Desc), vp, vp, vp, vp, sz, vp, sz, vp, sz, ctypes.POINTER(sz), vp]
        L.anslin_gemm_launches.restype = ctypes.c_int
        L.anslin_gemm_launches.argtypes = [ctypes.c_int64]
        L.anslin_status_string.argtypes = [ctypes.c_int]; L.anslin_status_string.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise AnslinError("%s failed: %s (status %d)" % (what, lib().anslin_status_string(rc).decode(), rc))


def _hp(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


def anslin_encode_host(fmt: int, w: np.ndarray, n_out: int, k_in: int, tile_k: int = 0, flags: int = 0,
                       scales: np.ndarray | None = None, zeros: np.ndarray | None = None, group_size: int = 0,
                       w_scale: float = 1.0, tile_n: int = 0):
    """Returns (container as np.uint8 array, stats dict)."""
    d = Desc(fmt, n_out, k_in, tile_k, group_size, flags, w_scale, tile_n)
    cap = lib().anslin_encode_bound(ctypes.byref(d))
    if cap == 0:
        raise AnslinError("anslin_encode_bound: unsupported shape or format")
    w = np.ascontiguousarray(w)
    scales = None if scales is None else np.ascontiguousarray(scales, dtype=np.float16)
    zeros = None if zeros is None else np.ascontiguousarray(zeros, dtype=np.float16)
    out = np.empty(cap, dtype=np.uint8)
    n = ctypes.c_size_t(0)
    st = Stats()
    _check(lib().anslin_encode_host(ctypes.byref(d), _hp(w), _hp(scales), _hp(zeros), _hp(out), cap, ctypes.byref(n),
                                    ctypes.byref(st)), "anslin_encode_host")
    return out[:n.value].copy(), st.as_dict()


def anslin_encode_device(fmt: int, w_ptr: int, n_out: int, k_in: int, container_ptr: int, capacity: int, ws_ptr: int, ws_bytes: int,
                         tile_k: int = 256, flags: int = FLAG_LANE_STREAMS, scales: np.ndarray | None = None,
                         zeros: np.ndarray | None = None, group_size: int = 0, w_scale: float = 1.0, stream: int = 0):
    """GPU-side encoder: W at w_ptr (device) -> container at container_ptr (device).  Returns (head bytes as np.uint8
    array = what Weight() needs as container_host, container size in bytes)."""
    d = Desc(fmt, n_out, k_in, tile_k, group_size, flags, w_scale, 32)
    hb = int(lib().anslin_encode_device_head_bytes(ctypes.byref(d)))
    if hb == 0:
        raise AnslinError("anslin_encode_device: unsupported geometry (lane streams, 32-row tiles, 256-step segments)")
    scales = None if scales is None else np.ascontiguousarray(scales, dtype=np.float16)
    zeros = None if zeros is None else np.ascontiguousarray(zeros, dtype=np.float16)
    head = np.zeros(hb, dtype=np.uint8)
    n = ctypes.c_size_t(0)
    _check(lib().anslin_encode_device(ctypes.byref(d), ctypes.c_void_p(w_ptr), _hp(scales), _hp(zeros), ctypes.c_void_p(container_ptr),
                                      capacity, _hp(head), hb, ctypes.c_void_p(ws_ptr), ws_bytes, ctypes.byref(n), ctypes.c_void_p(stream)),
           "anslin_encode_device")
    return head, int(n.value)


def anslin_encode_bound(fmt: int, n_out: int, k_in: int, tile_k: int = 0, flags: int = 0, group_size: int = 0, tile_n: int = 0) -> int:
    d = Desc(fmt, n_out, k_in, tile_k, group_size, flags, 1.0, tile_n)
    return int(lib().anslin_encode_bound(ctypes.byref(d)))


def anslin_encode_device_workspace_bytes(fmt: int, n_out: int, k_in: int, tile_k: int = 256, flags: int = FLAG_LANE_STREAMS,
                                         group_size: int = 0) -> int:
    d = Desc(fmt, n_out, k_in, tile_k, group_size, flags, 1.0, 32)
    return int(lib().anslin_encode_device_workspace_bytes(ctypes.byref(d)))


class Weight:
    """Host handle (anslin_weight*) bound to a device copy of the container."""

    def __init__(self, container_host: np.ndarray, container_dev_ptr: int | None):
        self._h = ctypes.c_void_p()
        c = np.ascontiguousarray(container_host, dtype=np.uint8)
        _check(lib().anslin_open(_hp(c), c.size, ctypes.c_void_p(container_dev_ptr or 0), ctypes.byref(self._h)), "anslin_open")
        d = Desc()
        _check(lib().anslin_describe(self._h, ctypes.byref(d)), "anslin_describe")
        self.desc = d
        self.nbytes = c.size

    @property
    def handle(self):
        return self._h

    def close(self):
        if self._h:
            lib().anslin_close(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def anslin_decode(w: Weight, out_ptr: int, capacity: int, stream: int = 0):
    _check(lib().anslin_decode(w.handle, ctypes.c_void_p(out_ptr), capacity, ctypes.c_void_p(stream)), "anslin_decode")


def anslin_gemm_workspace_bytes(w: Weight, m: int) -> int:
    return int(lib().anslin_gemm_workspace_bytes(w.handle, m))


def anslin_gemm(w: Weight, x_ptr: int, x_dtype: int, ldx: int, m: int, x_scale_ptr: int | None, y_ptr: int, ldy: int,
                ws_ptr: int, ws_bytes: int, stream: int = 0):
    _check(lib().anslin_gemm(w.handle, ctypes.c_void_p(x_ptr), x_dtype, ldx, m, ctypes.c_void_p(x_scale_ptr or 0),
                             ctypes.c_void_p(y_ptr), ldy, ctypes.c_void_p(ws_ptr), ws_bytes, ctypes.c_void_p(stream)), "anslin_gemm")


STATIC_WORKSPACE_BYTES = 24 << 20


def anslin_gemm_static(w: Weight, x_ptr: int, x_dtype: int, ldx: int, m: int, x_scale_ptr: int | None, y_ptr: int, ldy: int,
                       stream: int = 0):
    """anslin_gemm on the library's static workspace: allocates nothing (include/anslin.h)."""
    _check(lib().anslin_gemm_static(w.handle, ctypes.c_void_p(x_ptr), x_dtype, ldx, m, ctypes.c_void_p(x_scale_ptr or 0),
                                    ctypes.c_void_p(y_ptr), ldy, ctypes.c_void_p(stream)), "anslin_gemm_static")


def anslin_gemm_multi_workspace_bytes(weights, m_max: int) -> int:
    n = len(weights)
    arr = (ctypes.c_void_p * n)(*[w.handle for w in weights])
    return int(lib().anslin_gemm_multi_workspace_bytes(arr, n, int(m_max)))


class MultiCall:
    """Marshalled argument arrays of one anslin_gemm_multi call (built once, reusable every step)."""

    def __init__(self, weights, x_ptrs, x_dtype, ldxs, ms, x_scale_ptrs, y_ptrs, ldys, ws_ptr, ws_bytes, y_dtype: int = DT_F32):
        n = self.n = len(weights)
        self.y_dtype = y_dtype
        vp, i64, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32
        self.w = (vp * n)(*[w.handle for w in weights])
        self.x = (vp * n)(*[int(p) for p in x_ptrs])
        self.ldx = (i64 * n)(*[int(v) for v in ldxs])
        self.m = (i32 * n)(*[int(v) for v in ms])
        self.xs = None if x_scale_ptrs is None else (vp * n)(*[int(p or 0) for p in x_scale_ptrs])
        self.y = (vp * n)(*[int(p) for p in y_ptrs])
        self.ldy = (i64 * n)(*[int(v) for v in ldys])
        self.x_dtype, self.ws_ptr, self.ws_bytes = x_dtype, ctypes.c_void_p(ws_ptr), ws_bytes

    def __call__(self, stream: int = 0):
        _check(lib().anslin_gemm_multi_ex(self.w, self.n, self.x, self.x_dtype, self.ldx, self.m, self.xs, self.y, self.y_dtype, self.ldy,
                                          self.ws_ptr, self.ws_bytes, ctypes.c_void_p(stream)), "anslin_gemm_multi_ex")


def anslin_gemm_multi(weights, x_ptrs, x_dtype, ldxs, ms, x_scale_ptrs, y_ptrs, ldys, ws_ptr, ws_bytes, stream: int = 0):
    n = len(weights)
    c = MultiCall(weights, x_ptrs, x_dtype, ldxs, ms, x_scale_ptrs, y_ptrs, ldys, ws_ptr, ws_bytes)
    _check(lib().anslin_gemm_multi(c.w, n, c.x, c.x_dtype, c.ldx, c.m, c.xs, c.y, c.ldy, c.ws_ptr, c.ws_bytes, ctypes.c_void_p(stream)),
           "anslin_gemm_multi")


def anslin_gemm_multi_ex(weights, x_ptrs, x_dtype, ldxs, ms, x_scale_ptrs, y_ptrs, y_dtype, ldys, ws_ptr, ws_bytes, stream: int = 0):
    MultiCall(weights, x_ptrs, x_dtype, ldxs, ms, x_scale_ptrs, y_ptrs, ldys, ws_ptr, ws_bytes, y_dtype)(stream)


def anslin_gemm_grouped(experts, rows_per_expert, x_ptr: int, x_dtype: int, ldx: int, x_scale_ptr: int | None, y_ptr: int,
                        ldy: int, ws_ptr: int, ws_bytes: int, stream: int = 0):
    n = len(experts)
    arr = (ctypes.c_void_p * n)(*[e.handle for e in experts])
    rows = (ctypes.c_int32 * n)(*[int(r) for r in rows_per_expert])
    _check(lib().anslin_gemm_grouped(arr, n, rows, ctypes.c_void_p(x_ptr), x_dtype, ldx, ctypes.c_void_p(x_scale_ptr or 0),
                                     ctypes.c_void_p(y_ptr), ldy, ctypes.c_void_p(ws_ptr), ws_bytes, ctypes.c_void_p(stream)),
           "anslin_gemm_grouped")


def anslin_dense_workspace_bytes(n_out: int, k_in: int, m: int) -> int:
    return int(lib().anslin_dense_workspace_bytes(n_out, k_in, m))


def anslin_dense_gemm(fmt: int, w_ptr: int, n_out: int, k_in: int, w_scale_ptr: int | None, w_scale: float, x_ptr: int,
                      x_dtype: int, ldx: int, m: int, x_scale_ptr: int | None, y_ptr: int, ldy: int, ws_ptr: int, ws_bytes: int,
                      stream: int = 0):
    _check(lib().anslin_dense_gemm(fmt, ctypes.c_void_p(w_ptr), n_out, k_in, ctypes.c_void_p(w_scale_ptr or 0), w_scale,
                                   ctypes.c_void_p(x_ptr), x_dtype, ldx, m, ctypes.c_void_p(x_scale_ptr or 0),
                                   ctypes.c_void_p(y_ptr), ldy, ctypes.c_void_p(ws_ptr), ws_bytes, ctypes.c_void_p(stream)),
           "anslin_dense_gemm")


def anslin_histogram(fmt: int, w_ptr: int, n_elems: int, counts_ptr: int, stream: int = 0):
    _check(lib().anslin_histogram(fmt, ctypes.c_void_p(w_ptr), n_elems, ctypes.c_void_p(counts_ptr), ctypes.c_void_p(stream)),
           "anslin_histogram")


def anslin_entropy_bits(counts) -> float:
    c = np.ascontiguousarray(counts, dtype=np.uint64)
    return float(lib().anslin_entropy_bits(c.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)), c.size))


def anslin_entropy_weighted(hs, ns) -> float:
    h = np.ascontiguousarray(hs, dtype=np.float64)
    n = np.ascontiguousarray(ns, dtype=np.uint64)
    return float(lib().anslin_entropy_weighted(h.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                               n.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)), h.size))


def anslin_gemm_launches(row_blocks: int) -> int:
    return int(lib().anslin_gemm_launches(int(row_blocks)))
