"""Seeded synthetic inputs shaped like BASELINE.json's five configs.

This module serves BOTH the oracle-side tests and the CUDA path and therefore holds none of the
method's arithmetic (no histogram, no rANS, no GEMM): only random draws, dtype casts and the
quantisers that DEFINE the inputs (SQ8 per reading A14, AWQ-style per A13, fp8 per A15 of
DESIGN.md).  The paper's real checkpoints (P:l.339) are not available offline; these stand in.
"""
from __future__ import annotations

import numpy as np

FMT_BF16, FMT_FP8_E4M3, FMT_INT8, FMT_INT4_AWQ, FMT_FP8_E5M2, FMT_FP4_E2M1, FMT_BF16_PAIR4 = 0, 1, 2, 3, 4, 5, 6

# BASELINE.json configs 2/3 (Qwen-14B-shaped dense decoder layer), [n_out, k_in] = Linear.weight
QWEN14B_LAYER = [("q", 5120, 5120), ("k", 1024, 5120), ("v", 1024, 5120), ("o", 5120, 5120),
                 ("gate", 13824, 5120), ("up", 13824, 5120), ("down", 5120, 13824)]
# config 4 (Llama-70B-shaped FFN)
LLAMA70B_FFN = [("gate", 28672, 8192), ("up", 28672, 8192), ("down", 8192, 28672)]
# config 5 (Mixtral-8x22B-shaped expert FFN), 8 experts each
MIXTRAL_EXPERT = [("gate", 16384, 6144), ("up", 16384, 6144), ("down", 6144, 16384)]


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit patterns (uint16), round to nearest even."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + r) >> 16).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << 16).view(np.float32)


def weights_f32(n_out: int, k_in: int, seed: int, std: float = 0.02, jitter: bool = False,
                outliers: bool = True) -> np.ndarray:
    """N(0, std^2), optional per-output-channel std jitter U(0.5, 1.5), 0.1 % outlier entries x20."""
    rng = np.random.default_rng(seed)
    w = rng.standard_normal((n_out, k_in), dtype=np.float32) * np.float32(std)
    if jitter:
        w *= rng.uniform(0.5, 1.5, size=(n_out, 1)).astype(np.float32)
    if outliers:
        n = max(1, int(round(1e-3 * n_out * k_in)))
        idx = rng.integers(0, n_out * k_in, size=n)
        w.reshape(-1)[idx] *= np.float32(20.0)
    return w


def acts_f32(m: int, k_in: int, seed: int) -> np.ndarray:
    return np.random.default_rng(seed).standard_normal((m, k_in), dtype=np.float32)


def quant_sq8_weights(w: np.ndarray):
    """Per-output-channel symmetric int8 (A14): s = max|w|/127 rounded to fp16; q = clip(rint(w/s))."""
    s = (np.abs(w).max(axis=1) / 127.0).astype(np.float16)
    s = np.maximum(s, np.float16(6e-8))
    q = np.clip(np.rint(w / s.astype(np.float32)[:, None]), -127, 127).astype(np.int8)
    return q, s


def quant_int8_acts(x: np.ndarray):
    """Per-token symmetric int8: s = max|x|/127 (fp32)."""
    s = (np.abs(x).max(axis=1) / 127.0).astype(np.float32)
    s = np.maximum(s, np.float32(1e-12))
    q = np.clip(np.rint(x / s[:, None]), -127, 127).astype(np.int8)
    return q, s


def quant_awq4_weights(w: np.ndarray, group: int = 128):
    """AWQ-style group-wise 4-bit (A13): per (row, group) s = (max-min)/15, z = clip(rint(-min/s),0,15),
    q = clip(rint(w/s) + z, 0, 15); s and z stored as fp16.  Returns (packed uint8 [n x k/2] with the
    low nibble = even k, scales fp16 [n x k/group], zeros fp16 [n x k/group])."""
    n, k = w.shape
    g = w.reshape(n, k // group, group)
    lo, hi = g.min(axis=2), g.max(axis=2)
    s = ((hi - lo) / 15.0).astype(np.float16)
    s = np.maximum(s, np.float16(6e-8))
    sf = s.astype(np.float32)
    z = np.clip(np.rint(-lo / sf), 0, 15)
    q = np.clip(np.rint(g / sf[:, :, None]) + z[:, :, None], 0, 15).astype(np.uint8).reshape(n, k)
    packed = (q[:, 0::2] | (q[:, 1::2] << 4)).astype(np.uint8)
    return packed, s, z.astype(np.float16)


def quant_int4_sym_weights(w: np.ndarray):
    """Plain symmetric per-channel int4 (S: §8(f) NEXT-2 "plain int4"): s[n] = amax_n/7, q = clip(rint(w/s), -8, 7),
    stored offset-binary (q + 8) so that it IS the AWQ container with one group per row and zero point 8.
    Returns (packed uint8 [n x k/2], scales fp16 [n x 1], zeros fp16 [n x 1] = 8)."""
    n, k = w.shape
    s = np.maximum((np.abs(w).max(axis=1) / 7.0).astype(np.float16), np.float16(6e-8))
    q = (np.clip(np.rint(w / s.astype(np.float32)[:, None]), -8, 7) + 8).astype(np.uint8)
    packed = (q[:, 0::2] | (q[:, 1::2] << 4)).astype(np.uint8)
    return packed, s.reshape(n, 1), np.full((n, 1), 8, dtype=np.float16)


def f32_to_e4m3_bytes(x: np.ndarray) -> np.ndarray:
    """float32 -> OCP e4m3fn byte codes via torch's CPU cast (round to nearest even, saturating inputs
    are the caller's job: values are pre-scaled to |x| <= 448)."""
    import torch
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(torch.float8_e4m3fn)
    return t.view(torch.uint8).numpy().copy()


def quant_fp8_weights(w: np.ndarray):
    """Per-tensor e4m3 (A15): s = amax/448."""
    s = float(np.abs(w).max() / 448.0)
    return f32_to_e4m3_bytes(w / np.float32(s)), s


def quant_fp8_acts(x: np.ndarray):
    """Per-token e4m3: s[m] = amax_m/448 (fp32)."""
    s = (np.abs(x).max(axis=1) / 448.0).astype(np.float32)
    s = np.maximum(s, np.float32(1e-12))
    return f32_to_e4m3_bytes(x / s[:, None]), s


def f32_to_e5m2_bytes(x: np.ndarray) -> np.ndarray:
    """float32 -> OCP e5m2 byte codes via torch's CPU cast (values pre-scaled to |x| <= 57344)."""
    import torch
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).to(torch.float8_e5m2)
    return t.view(torch.uint8).numpy().copy()


def quant_fp8_e5m2_weights(w: np.ndarray):
    """Per-tensor e5m2: s = amax/57344 (the largest finite e5m2), same recipe as A15."""
    s = float(np.abs(w).max() / 57344.0)
    return f32_to_e5m2_bytes(w / np.float32(s)), s


def quant_fp8_e5m2_acts(x: np.ndarray):
    """Per-token e5m2: s[m] = amax_m/57344 (fp32)."""
    s = (np.abs(x).max(axis=1) / 57344.0).astype(np.float32)
    s = np.maximum(s, np.float32(1e-12))
    return f32_to_e5m2_bytes(x / s[:, None]), s


def quant_fp4_weights(w: np.ndarray):
    """Per-tensor fp4-e2m1: s = amax/6, every w/s rounded to the nearest of the 8 magnitudes
    0, 0.5, 1, 1.5, 2, 3, 4, 6 (ties to the even code), sign in bit 3.  Returns (packed uint8 [n x k/2], s)."""
    s = float(np.abs(w).max() / 6.0)
    grid = np.array([0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0], dtype=np.float32)
    a = np.abs(w / np.float32(s)).astype(np.float32)
    hi = np.clip(np.searchsorted(grid, a, side="left"), 1, 7)
    lo = hi - 1
    d_lo, d_hi = a - grid[lo], grid[hi] - a
    code = np.where(d_lo < d_hi, lo, np.where(d_hi < d_lo, hi, np.where(lo % 2 == 0, lo, hi))).astype(np.uint8)
    code |= (np.signbit(w).astype(np.uint8) << 3)
    return (code[:, 0::2] | (code[:, 1::2] << 4)).astype(np.uint8), s


def route_top2(m_tokens: int, n_experts: int, seed: int):
    """Uniform-random router logits -> top-2 experts per token (tie -> lower id).  Returns
    (rows_per_expert int32 [E], token index of every row, sorted by expert) (A17)."""
    rng = np.random.default_rng(seed)
    logits = rng.uniform(size=(m_tokens, n_experts))
    top = np.argsort(-logits, axis=1, kind="stable")[:, :2]
    tok = np.repeat(np.arange(m_tokens), 2)
    exp = top.reshape(-1)
    order = np.argsort(exp, kind="stable")
    rows = np.bincount(exp, minlength=n_experts).astype(np.int32)
    return rows, tok[order]


def config1():
    """BASELINE config 1: W 1024x1024 bf16 N(0,0.02^2) + 0.1 % outliers x20 (seed 0), X 8x1024 bf16 N(0,1)."""
    w = f32_to_bf16_bits(weights_f32(1024, 1024, seed=0))
    x = f32_to_bf16_bits(acts_f32(8, 1024, seed=1000))
    return w, x
