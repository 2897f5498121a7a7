"""ORACLE (test infrastructure only) — reference GEMM Y = X . W^T in float64 / int64.

The method reaches exactly the plain definition Y[m,n] = sum_k X[m,k] * W[n,k] (P:l.310 §V-E,
Alg V.3 P:l.301-304) over losslessly reconstructed weights, so the oracle IS that definition:
inputs converted exactly to float64, one library matmul, no blocking.  Also returns
A[m,n] = sum_k |X[m,k] * W[n,k]|, the scale of BASELINE.json's per-element tolerance.
"""
from __future__ import annotations

import numpy as np


def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    """bf16 is the upper half of an IEEE float32."""
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def e4m3_to_f64(code: np.ndarray) -> np.ndarray:
    """OCP FP8 E4M3 (the 'fn' flavour: bias 7, no infinities, S.1111.111 = NaN), written out from
    the format definition: (-1)^s * 2^(e-7) * (1 + m/8), subnormals 2^-6 * m/8."""
    c = code.view(np.uint8).astype(np.int64)
    s = (c >> 7) & 1
    e = (c >> 3) & 0xF
    m = c & 7
    val = np.where(e == 0, np.ldexp(m / 8.0, -6), np.ldexp(1.0 + m / 8.0, e - 7))
    val = np.where((e == 15) & (m == 7), np.nan, val)
    return np.where(s == 1, -val, val)


def e5m2_to_f64(code: np.ndarray) -> np.ndarray:
    """OCP FP8 E5M2 (P:l.80): IEEE-like, bias 15: (-1)^s * 2^(e-15) * (1 + m/4), subnormals 2^-14 * m/4,
    e = 31: infinity (m = 0) or NaN.  It is the upper byte of an IEEE binary16."""
    c = code.view(np.uint8).astype(np.int64)
    s = (c >> 7) & 1
    e = (c >> 2) & 0x1F
    m = c & 3
    val = np.where(e == 0, np.ldexp(m / 4.0, -14), np.ldexp(1.0 + m / 4.0, e - 15))
    val = np.where(e == 31, np.where(m == 0, np.inf, np.nan), val)
    return np.where(s == 1, -val, val)


def e2m1_to_f64(code: np.ndarray) -> np.ndarray:
    """OCP FP4 E2M1 (P:l.80), 4-bit codes s.ee.m, bias 1: (-1)^s * 2^(e-1) * (1 + m/2), subnormal (e = 0) m/2;
    no infinities or NaNs: magnitudes 0, 0.5, 1, 1.5, 2, 3, 4, 6."""
    c = code.astype(np.int64)
    s = (c >> 3) & 1
    e = (c >> 1) & 3
    m = c & 1
    val = np.where(e == 0, m / 2.0, np.ldexp(1.0 + m / 2.0, e - 1))
    return np.where(s == 1, -val, val)


def int4_unpack(packed: np.ndarray) -> np.ndarray:
    """uint8 [n x k/2], low nibble = even k  ->  uint8 [n x k] codes 0..15."""
    p = packed.view(np.uint8)
    out = np.zeros((p.shape[0], p.shape[1] * 2), dtype=np.uint8)
    out[:, 0::2] = p & 0xF
    out[:, 1::2] = p >> 4
    return out


def awq_dequant_f64(packed: np.ndarray, scales: np.ndarray, zeros: np.ndarray, group: int) -> np.ndarray:
    """w = (q - z) * s evaluated exactly in float64 from the fp16-valued s and z (reading A13)."""
    q = int4_unpack(packed).astype(np.float64)
    s = np.repeat(scales.astype(np.float64), group, axis=1)
    z = np.repeat(zeros.astype(np.float64), group, axis=1)
    return (q - z) * s


def gemm_f64(x: np.ndarray, w: np.ndarray):
    """x [M x K], w [N x K] float64 -> (Y, A) float64."""
    return x @ w.T, np.abs(x) @ np.abs(w).T


def gemm_bf16(x_bits: np.ndarray, w_bits: np.ndarray):
    return gemm_f64(bf16_bits_to_f64(x_bits), bf16_bits_to_f64(w_bits))


def gemm_int8(xq: np.ndarray, x_scale: np.ndarray, wq: np.ndarray, w_scale: np.ndarray):
    """SQ8 (reading A14): int64 accumulate, then * s_x[m] * s_w[n] in float64.
    Returns (Y, A, acc) with acc the exact integer sums."""
    acc = xq.astype(np.int64) @ wq.astype(np.int64).T
    sc = x_scale.astype(np.float64)[:, None] * w_scale.astype(np.float64)[None, :]
    a = (np.abs(xq.astype(np.int64)) @ np.abs(wq.astype(np.int64)).T).astype(np.float64) * sc
    return acc.astype(np.float64) * sc, a, acc


def gemm_fp8(xq: np.ndarray, x_scale: np.ndarray, wq: np.ndarray, w_scale: float, x_e5m2: bool = False, w_e5m2: bool = False):
    """fp8 (reading A15): Y = (sum_k x8*w8) * s_x[m] * s_w; each operand e4m3 unless flagged e5m2."""
    y, a = gemm_f64((e5m2_to_f64 if x_e5m2 else e4m3_to_f64)(xq), (e5m2_to_f64 if w_e5m2 else e4m3_to_f64)(wq))
    sc = x_scale.astype(np.float64)[:, None] * float(w_scale)
    return y * sc, a * sc


def gemm_fp4(xq: np.ndarray, x_scale: np.ndarray, packed: np.ndarray, w_scale: float, x_e5m2: bool = False):
    """fp4-e2m1 weights (two codes per byte, low nibble = even k), fp8 activations with per-token scales:
    Y = (sum_k x8 * w4) * s_x[m] * s_w, the fp8 recipe of A15 with the 4-bit value set."""
    y, a = gemm_f64((e5m2_to_f64 if x_e5m2 else e4m3_to_f64)(xq), e2m1_to_f64(int4_unpack(packed)))
    sc = x_scale.astype(np.float64)[:, None] * float(w_scale)
    return y * sc, a * sc


def gemm_int4(x_f16: np.ndarray, packed: np.ndarray, scales: np.ndarray, zeros: np.ndarray, group: int):
    return gemm_f64(x_f16.astype(np.float64), awq_dequant_f64(packed, scales, zeros, group))
