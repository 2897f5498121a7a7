"""ORACLE (test infrastructure only) — ctypes binding of oracle/anslin_oracle.c.

The arithmetic lives in the plain C file (one function per passage of the paper, cited there);
this module only marshals numpy arrays.  Nothing here may be imported by the product package
``paper_2606_15789_b200``; only tests/, ``__graft_entry__.smoke()`` and bench.py's cpu_baseline /
``--impl reference`` legs use it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "anslin_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, -O2).  Returns the path of the shared object."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        u8p, u16p, u32p, u64p = (ctypes.POINTER(t) for t in (ctypes.c_uint8, ctypes.c_uint16, ctypes.c_uint32, ctypes.c_uint64))
        sz, ci, u64, dbl = ctypes.c_size_t, ctypes.c_int, ctypes.c_uint64, ctypes.c_double
        L.orc_histogram.argtypes = [u8p, sz, u64p]; L.orc_histogram.restype = None
        L.orc_entropy.argtypes = [u64p, ci]; L.orc_entropy.restype = dbl
        L.orc_cross_entropy.argtypes = [u64p, u32p, ci, ci]; L.orc_cross_entropy.restype = dbl
        L.orc_normalize.argtypes = [u64p, ci, ci, u32p]; L.orc_normalize.restype = ci
        L.orc_cumulative.argtypes = [u32p, ci, u32p]; L.orc_cumulative.restype = None
        L.orc_slot_table.argtypes = [u32p, u32p, ci, ci, u8p]; L.orc_slot_table.restype = None
        L.orc_encode_scalar.argtypes = [u8p, sz, u32p, u32p, ci, ci, ci, u64, u64p, u16p]; L.orc_encode_scalar.restype = sz
        L.orc_decode_scalar.argtypes = [u64, u16p, sz, u32p, u32p, u8p, ci, ci, ci, u8p, u64p]; L.orc_decode_scalar.restype = sz
        L.orc_tile_encode.argtypes = [u8p, sz, ci, u32p, u32p, ci, ci, ci, u64p, u64p, u16p]; L.orc_tile_encode.restype = sz
        L.orc_encode_scalar_lit.argtypes = [u8p, sz, u32p, u32p, ci, ci, ci, u64, u16p, u64p, u16p, u32p]; L.orc_encode_scalar_lit.restype = sz
        L.orc_decode_scalar_lit.argtypes = [u64, u16p, sz, u32p, u32p, u8p, ci, ci, ci, u8p, u16p, u64p]; L.orc_decode_scalar_lit.restype = sz
        L.orc_tile_decode.argtypes = [u64p, u16p, sz, ci, u32p, u32p, u8p, ci, ci, ci, u8p, u64p]; L.orc_tile_decode.restype = sz
        L.orc_tile_encode_by_simulation.argtypes = [u8p, sz, ci, u32p, u32p, u8p, ci, ci, ci, u64p, u64p, u16p]
        L.orc_tile_encode_by_simulation.restype = sz
        _lib = L
    return _lib


def _p(a: np.ndarray, t):
    return a.ctypes.data_as(ctypes.POINTER(t))


def histogram(sym: np.ndarray) -> np.ndarray:
    sym = np.ascontiguousarray(sym, dtype=np.uint8).ravel()
    cnt = np.zeros(256, dtype=np.uint64)
    lib().orc_histogram(_p(sym, ctypes.c_uint8), sym.size, _p(cnt, ctypes.c_uint64))
    return cnt


def entropy(cnt: np.ndarray) -> float:
    cnt = np.ascontiguousarray(cnt, dtype=np.uint64)
    return float(lib().orc_entropy(_p(cnt, ctypes.c_uint64), cnt.size))


def cross_entropy(cnt: np.ndarray, f: np.ndarray, b: int) -> float:
    cnt = np.ascontiguousarray(cnt, dtype=np.uint64)
    f = np.ascontiguousarray(f, dtype=np.uint32)
    return float(lib().orc_cross_entropy(_p(cnt, ctypes.c_uint64), _p(f, ctypes.c_uint32), cnt.size, b))


def normalize(cnt: np.ndarray, b: int) -> np.ndarray:
    cnt = np.ascontiguousarray(cnt, dtype=np.uint64)
    f = np.zeros(cnt.size, dtype=np.uint32)
    rc = lib().orc_normalize(_p(cnt, ctypes.c_uint64), cnt.size, b, _p(f, ctypes.c_uint32))
    if rc != 0:
        raise ValueError("histogram cannot be normalised to 2^%d slots" % b)
    return f


def cumulative(f: np.ndarray) -> np.ndarray:
    f = np.ascontiguousarray(f, dtype=np.uint32)
    c = np.zeros(f.size, dtype=np.uint32)
    lib().orc_cumulative(_p(f, ctypes.c_uint32), f.size, _p(c, ctypes.c_uint32))
    return c


def slot_table(f: np.ndarray, c: np.ndarray, b: int) -> np.ndarray:
    f = np.ascontiguousarray(f, dtype=np.uint32)
    c = np.ascontiguousarray(c, dtype=np.uint32)
    if int(f.sum()) != (1 << b):
        raise ValueError("frequencies must sum to 2^b")
    t = np.zeros(1 << b, dtype=np.uint8)
    lib().orc_slot_table(_p(f, ctypes.c_uint32), _p(c, ctypes.c_uint32), f.size, b, _p(t, ctypes.c_uint8))
    return t


class Table:
    """Frequencies f, cumulative c and slot->symbol map for one codebook (P:l.149, l.271)."""

    def __init__(self, f: np.ndarray, b: int):
        self.b = b
        self.f = np.ascontiguousarray(f, dtype=np.uint32)
        self.c = cumulative(self.f)
        self.slots = slot_table(self.f, self.c, b)


def encode_scalar(sym, tab: Table, w: int, Llog2: int, x_init: int):
    sym = np.ascontiguousarray(sym, dtype=np.uint8)
    words = np.zeros(sym.size * 2 + 8, dtype=np.uint16)
    st = ctypes.c_uint64(0)
    n = lib().orc_encode_scalar(_p(sym, ctypes.c_uint8), sym.size, _p(tab.f, ctypes.c_uint32), _p(tab.c, ctypes.c_uint32),
                                tab.b, w, Llog2, x_init, ctypes.byref(st), _p(words, ctypes.c_uint16))
    return int(st.value), words[:n].copy()


def decode_scalar(state: int, words, n: int, tab: Table, w: int, Llog2: int):
    words = np.ascontiguousarray(np.concatenate([np.asarray(words, dtype=np.uint16), np.zeros(4, np.uint16)]))
    out = np.zeros(n, dtype=np.uint8)
    end = ctypes.c_uint64(0)
    used = lib().orc_decode_scalar(state, _p(words, ctypes.c_uint16), n, _p(tab.f, ctypes.c_uint32), _p(tab.c, ctypes.c_uint32),
                                   _p(tab.slots, ctypes.c_uint8), tab.b, w, Llog2, _p(out, ctypes.c_uint8), ctypes.byref(end))
    return out, int(end.value), int(used)


def encode_scalar_lit(sym, tab: Table, w: int, Llog2: int, x_init: int, lit):
    """Scalar stream whose symbols are pairs of 4-bit codes; code 15 = escape with an in-stream literal word
    (see orc_encode_scalar_lit).  Returns (start state, words in read order, words consumed after each step)."""
    sym = np.ascontiguousarray(sym, dtype=np.uint8)
    lit = np.ascontiguousarray(np.concatenate([np.asarray(lit, dtype=np.uint16), np.zeros(1, np.uint16)]))
    words = np.zeros(sym.size * 4 + 8, dtype=np.uint16)
    after = np.zeros(sym.size, dtype=np.uint32)
    st = ctypes.c_uint64(0)
    n = lib().orc_encode_scalar_lit(_p(sym, ctypes.c_uint8), sym.size, _p(tab.f, ctypes.c_uint32), _p(tab.c, ctypes.c_uint32),
                                    tab.b, w, Llog2, x_init, _p(lit, ctypes.c_uint16), ctypes.byref(st), _p(words, ctypes.c_uint16),
                                    _p(after, ctypes.c_uint32))
    return int(st.value), words[:n].copy(), after


def decode_scalar_lit(state: int, words, n: int, tab: Table, w: int, Llog2: int):
    """Returns (symbols, literal per nibble [2n] with 0xFFFF = none, end state, words consumed)."""
    words = np.ascontiguousarray(np.concatenate([np.asarray(words, dtype=np.uint16), np.zeros(4, np.uint16)]))
    out = np.zeros(n, dtype=np.uint8)
    lit = np.zeros(2 * n, dtype=np.uint16)
    end = ctypes.c_uint64(0)
    used = lib().orc_decode_scalar_lit(state, _p(words, ctypes.c_uint16), n, _p(tab.f, ctypes.c_uint32), _p(tab.c, ctypes.c_uint32),
                                       _p(tab.slots, ctypes.c_uint8), tab.b, w, Llog2, _p(out, ctypes.c_uint8), _p(lit, ctypes.c_uint16),
                                       ctypes.byref(end))
    return out, lit, int(end.value), int(used)


def tile_encode(sym, R: int, tab: Table, w: int, Llog2: int, x_init, by_simulation: bool = False):
    """sym is in tile order (symbol i -> lane i mod R, step i div R).  Returns (states[R], words)."""
    sym = np.ascontiguousarray(sym, dtype=np.uint8)
    assert sym.size % R == 0
    x_init = np.ascontiguousarray(np.broadcast_to(np.asarray(x_init, dtype=np.uint64), (R,)))
    states = np.zeros(R, dtype=np.uint64)
    words = np.zeros(sym.size * 2 + 8, dtype=np.uint16)
    if by_simulation:
        n = lib().orc_tile_encode_by_simulation(_p(sym, ctypes.c_uint8), sym.size, R, _p(tab.f, ctypes.c_uint32),
                                                _p(tab.c, ctypes.c_uint32), _p(tab.slots, ctypes.c_uint8), tab.b, w, Llog2,
                                                _p(x_init, ctypes.c_uint64), _p(states, ctypes.c_uint64), _p(words, ctypes.c_uint16))
    else:
        n = lib().orc_tile_encode(_p(sym, ctypes.c_uint8), sym.size, R, _p(tab.f, ctypes.c_uint32), _p(tab.c, ctypes.c_uint32),
                                  tab.b, w, Llog2, _p(x_init, ctypes.c_uint64), _p(states, ctypes.c_uint64), _p(words, ctypes.c_uint16))
    return states, words[:n].copy()


def tile_decode(states, words, n: int, R: int, tab: Table, w: int, Llog2: int):
    """Returns (symbols in tile order, end states[R], words consumed)."""
    states = np.ascontiguousarray(states, dtype=np.uint64)
    words = np.ascontiguousarray(np.concatenate([np.asarray(words, dtype=np.uint16), np.zeros(4, np.uint16)]))
    out = np.zeros(n, dtype=np.uint8)
    end = np.zeros(R, dtype=np.uint64)
    used = lib().orc_tile_decode(_p(states, ctypes.c_uint64), _p(words, ctypes.c_uint16), n, R, _p(tab.f, ctypes.c_uint32),
                                 _p(tab.c, ctypes.c_uint32), _p(tab.slots, ctypes.c_uint8), tab.b, w, Llog2,
                                 _p(out, ctypes.c_uint8), _p(end, ctypes.c_uint64))
    return out, end, int(used)
