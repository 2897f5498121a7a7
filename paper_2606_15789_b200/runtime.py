"""Device-memory plumbing around the C ABI: torch owns HBM buffers and streams, nothing else.

No arithmetic of the method happens here; every call forwards to libanslin through binding.py.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B

_TORCH_X = {B.FMT_BF16: torch.bfloat16, B.FMT_BF16_PAIR4: torch.bfloat16, B.FMT_INT4_AWQ: torch.float16, B.FMT_INT8: torch.int8,
            B.FMT_FP8_E4M3: torch.uint8, B.FMT_FP8_E5M2: torch.uint8, B.FMT_FP4_E2M1: torch.uint8}


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def x_to_device(fmt: int, x: np.ndarray) -> torch.Tensor:
    """numpy activations in the format's X dtype (bf16 as uint16 bits, fp16, int8, e4m3 bytes) -> cuda tensor."""
    t = torch.from_numpy(np.ascontiguousarray(x))
    if fmt == B.FMT_BF16:
        t = t.view(torch.int16).view(torch.bfloat16)
    return t.cuda()


class DeviceWeight:
    """A compressed weight matrix resident in HBM + its anslin_weight handle."""

    def __init__(self, container: np.ndarray, device: str = "cuda"):
        if not torch.cuda.is_available():
            raise B.AnslinError("no CUDA device: anslin has no CPU fallback")
        self.container_host = np.ascontiguousarray(container, dtype=np.uint8)
        self.container_dev = torch.from_numpy(self.container_host).to(device)
        self.weight = B.Weight(self.container_host, self.container_dev.data_ptr())
        d = self.weight.desc
        self.fmt, self.n_out, self.k_in = d.format, d.n_out, d.k_in
        self._ws = None

    def close(self):
        self.weight.close()

    def decode(self) -> torch.Tensor:
        """anslin_decode -> row-major W in its original dtype/packing (bf16 as int16 bit patterns)."""
        if self.fmt in (B.FMT_BF16, B.FMT_BF16_PAIR4):
            out = torch.empty((self.n_out, self.k_in), dtype=torch.int16, device=self.container_dev.device)
        elif self.fmt in (B.FMT_INT4_AWQ, B.FMT_FP4_E2M1):
            out = torch.empty((self.n_out, self.k_in // 2), dtype=torch.uint8, device=self.container_dev.device)
        else:
            out = torch.empty((self.n_out, self.k_in), dtype=torch.uint8, device=self.container_dev.device)
        B.anslin_decode(self.weight, out.data_ptr(), out.numel() * out.element_size(), _stream())
        return out

    def workspace(self, m: int) -> torch.Tensor:
        need = B.anslin_gemm_workspace_bytes(self.weight, m)
        if self._ws is None or self._ws.numel() < need:
            self._ws = torch.empty(need, dtype=torch.uint8, device=self.container_dev.device)
        return self._ws

    def gemm(self, x: torch.Tensor, x_scale: torch.Tensor | None = None, y: torch.Tensor | None = None,
             x_dtype: int | None = None) -> torch.Tensor:
        """anslin_gemm: Y[m x n_out] f32 = X . W^T with W decoded on the fly (x_dtype: B.DT_*, default the format's own)."""
        m = x.shape[0]
        if y is None:
            y = torch.empty((m, self.n_out), dtype=torch.float32, device=x.device)
        ws = self.workspace(m)
        B.anslin_gemm(self.weight, x.data_ptr(), B.X_DTYPE[self.fmt] if x_dtype is None else x_dtype, x.stride(0), m,
                      None if x_scale is None else x_scale.data_ptr(), y.data_ptr(), y.stride(0), ws.data_ptr(), ws.numel(), _stream())
        return y


    def gemm_static(self, x: torch.Tensor, x_scale: torch.Tensor | None = None, y: torch.Tensor | None = None,
                    x_dtype: int | None = None) -> torch.Tensor:
        """anslin_gemm_static: the same product on the library's static workspace; the call allocates nothing (y given)."""
        m = x.shape[0]
        if y is None:
            y = torch.empty((m, self.n_out), dtype=torch.float32, device=x.device)
        B.anslin_gemm_static(self.weight, x.data_ptr(), B.X_DTYPE[self.fmt] if x_dtype is None else x_dtype, x.stride(0), m,
                             None if x_scale is None else x_scale.data_ptr(), y.data_ptr(), y.stride(0), _stream())
        return y

def encode_on_device(fmt: int, w: torch.Tensor, n_out: int, k_in: int, tile_k: int = 256, flags: int = B.FLAG_LANE_STREAMS,
                     scales: np.ndarray | None = None, zeros: np.ndarray | None = None, group_size: int = 0,
                     w_scale: float = 1.0) -> "DeviceWeight":
    """anslin_encode_device: compress a cuda tensor W (stored elements, row-major) without moving it to the host.
    Returns a DeviceWeight whose container lives in a device buffer trimmed to the container size."""
    cap = B.anslin_encode_bound(fmt, n_out, k_in, tile_k, flags, group_size, 32)
    need = B.anslin_encode_device_workspace_bytes(fmt, n_out, k_in, tile_k, flags, group_size)
    if cap == 0 or need == 0:
        raise B.AnslinError("encode_on_device: unsupported geometry")
    w = w.contiguous()
    out = torch.empty(cap, dtype=torch.uint8, device=w.device)
    ws = torch.empty(need, dtype=torch.uint8, device=w.device)
    head, n = B.anslin_encode_device(fmt, w.data_ptr(), n_out, k_in, out.data_ptr(), cap, ws.data_ptr(), need, tile_k=tile_k,
                                     flags=flags, scales=scales, zeros=zeros, group_size=group_size, w_scale=w_scale, stream=_stream())
    dw = DeviceWeight.__new__(DeviceWeight)
    dw.container_host = head
    dw.container_dev = out[:n]
    dw.weight = B.Weight(head, out.data_ptr())
    d = dw.weight.desc
    dw.fmt, dw.n_out, dw.k_in = d.format, d.n_out, d.k_in
    dw._ws = None
    return dw


class MultiGemm:
    """anslin_gemm_multi over weights that share format and tile geometry: ONE persistent launch for
    e.g. q/k/v (same X) or gate/up.  Buffers and the marshalled call are built once."""

    def __init__(self, dws, xs, x_scales=None, ys=None, y_dtype: torch.dtype = torch.float32):
        self.dws, self.xs = list(dws), list(xs)
        dev = self.xs[0].device
        ms = [int(x.shape[0]) for x in self.xs]
        self.ys = list(ys) if ys is not None else [torch.empty((m, d.n_out), dtype=y_dtype, device=dev)
                                                   for m, d in zip(ms, self.dws)]
        ydt = {torch.float32: B.DT_F32, torch.bfloat16: B.DT_BF16}[self.ys[0].dtype]
        assert all(y.dtype == self.ys[0].dtype for y in self.ys)
        self.x_scales = x_scales
        need = B.anslin_gemm_multi_workspace_bytes([d.weight for d in self.dws], max(ms))
        self.ws = torch.empty(need, dtype=torch.uint8, device=dev)
        self.call = B.MultiCall([d.weight for d in self.dws], [x.data_ptr() for x in self.xs], B.X_DTYPE[self.dws[0].fmt],
                                [x.stride(0) for x in self.xs], ms,
                                None if x_scales is None else [s.data_ptr() for s in x_scales],
                                [y.data_ptr() for y in self.ys], [y.stride(0) for y in self.ys], self.ws.data_ptr(), self.ws.numel(), ydt)

    def __call__(self):
        self.call(_stream())
        return self.ys


def gemm_grouped(experts, rows_per_expert, x: torch.Tensor, x_scale: torch.Tensor | None, y: torch.Tensor | None = None):
    m = x.shape[0]
    if y is None:
        y = torch.empty((m, experts[0].n_out), dtype=torch.float32, device=x.device)
    blocks = sum((int(r) + 255) // 256 for r in rows_per_expert)     # experts with > 256 rows run as several problems
    per_launch = [experts[0].weight] * max(1, min(8, blocks)) if blocks > len(experts) else [e.weight for e in experts]
    need = B.anslin_gemm_multi_workspace_bytes(per_launch, int(min(256, max(max(rows_per_expert), 1))))
    ws = experts[0]._ws
    if ws is None or ws.numel() < need:
        ws = experts[0]._ws = torch.empty(need, dtype=torch.uint8, device=x.device)
    B.anslin_gemm_grouped([e.weight for e in experts], rows_per_expert, x.data_ptr(), B.X_DTYPE[experts[0].fmt], x.stride(0),
                          None if x_scale is None else x_scale.data_ptr(), y.data_ptr(), y.stride(0), ws.data_ptr(), ws.numel(), _stream())
    return y


def dense_gemm(fmt: int, w: torch.Tensor, x: torch.Tensor, w_scale_vec: torch.Tensor | None = None, w_scale: float = 1.0,
               x_scale: torch.Tensor | None = None, y: torch.Tensor | None = None, ws: torch.Tensor | None = None):
    """Uncompressed comparator (anslin_dense_gemm): w is row-major W in the operand dtype."""
    n_out, k_in = w.shape
    m = x.shape[0]
    if y is None:
        y = torch.empty((m, n_out), dtype=torch.float32, device=x.device)
    if ws is None:
        ws = torch.empty(B.anslin_dense_workspace_bytes(n_out, k_in, m), dtype=torch.uint8, device=x.device)
    B.anslin_dense_gemm(fmt, w.data_ptr(), n_out, k_in, None if w_scale_vec is None else w_scale_vec.data_ptr(), w_scale,
                        x.data_ptr(), B.X_DTYPE[fmt], x.stride(0), m, None if x_scale is None else x_scale.data_ptr(),
                        y.data_ptr(), y.stride(0), ws.data_ptr(), ws.numel(), _stream())
    return y


# Tile geometries the library supports (tile_n, tile_k, layout flags), tried by autotune_tile.
TILE_CANDIDATES = ((128, 64, 0), (128, 128, 0), (128, 256, 0), (32, 128, 0), (32, 256, 0), (32, 256, B.FLAG_LANE_STREAMS),
                   (32, 512, B.FLAG_LANE_STREAMS), (32, 1024, B.FLAG_LANE_STREAMS))


def autotune_tile(fmt: int, w: np.ndarray, n_out: int, k_in: int, m: int, x: torch.Tensor, x_scale: torch.Tensor | None = None,
                  candidates=TILE_CANDIDATES, iters: int = 20, max_gap_bits: float | None = None, **encode_kw):
    """Per-matrix choice of the tile geometry (P:l.167 "profiled to determine the optimal tensor-core tiling
    geometry"; S: §8(f) NEXT-2): encode W with every candidate (tile_n, tile_k, layout flags) that fits the
    shape, time anslin_gemm at batch size m with CUDA events, and return
    (best, rows) -- best = dict(tile_n, tile_k, flags, us, bits_per_weight, container) of the fastest candidate
    whose bits/weight is within max_gap_bits of the smallest one seen (None = no size constraint), rows = one
    dict per candidate tried.  Measurement only: all arithmetic runs in the library."""
    base_flags = int(encode_kw.pop("flags", 0))
    rows = []
    for tile_n, tile_k, lflags in candidates:
        if k_in % tile_k or n_out % 128:
            continue
        try:
            buf, st = B.anslin_encode_host(fmt, w, n_out, k_in, tile_k=tile_k, tile_n=tile_n, flags=base_flags | lflags, **encode_kw)
        except B.AnslinError:
            continue          # geometry not supported for this format
        dw = DeviceWeight(buf)
        y = torch.empty((m, n_out), dtype=torch.float32, device=x.device)
        for _ in range(3):
            dw.gemm(x, x_scale, y)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(iters):
            dw.gemm(x, x_scale, y)
        e1.record()
        e1.synchronize()
        rows.append(dict(tile_n=tile_n, tile_k=tile_k, flags=int(dw.weight.desc.flags), us=e0.elapsed_time(e1) * 1e3 / iters,
                         bits_per_weight=st["bits_per_weight"], container=buf))
        dw.close()
    if not rows:
        raise B.AnslinError("autotune_tile: no candidate geometry fits this shape")
    smallest = min(r["bits_per_weight"] for r in rows)
    ok = [r for r in rows if max_gap_bits is None or r["bits_per_weight"] <= smallest + max_gap_bits]
    return min(ok, key=lambda r: r["us"]), rows


def entropy_study(fmt: int, tensors):
    """P:l.64-78 entropy study over device-resident weight tensors of one numeric format (S: NEXT-4): per tensor the
    256-bin histograms (anslin_histogram) and their entropies, and the symbol-weighted model entropy (P:l.74).
    tensors: cuda tensors of the stored elements (bf16 as int16/bfloat16, others as bytes).  Returns
    dict(layers=[dict(n_weights, counts[2][256], h_coded, h_side, bits_per_weight)], model_bits_per_weight);
    bits_per_weight = H(exponent) + H(sign|mantissa) for bf16, H(byte) for fp8/int8, H(packed byte)/2 for int4/fp4
    (h_side for those: the entropy of the single 4-bit code, the symbol Fig. 2 counts)."""
    packed4 = fmt in (B.FMT_INT4_AWQ, B.FMT_FP4_E2M1)
    layers, counts_dev = [], []
    for t in tensors:
        t = t.contiguous()
        c = torch.empty((2, 256), dtype=torch.int64, device=t.device)
        B.anslin_histogram(fmt, t.data_ptr(), t.numel(), c.data_ptr(), _stream())
        counts_dev.append((t.numel(), c))
    for n, c in counts_dev:
        counts = c.cpu().numpy().astype(np.uint64)
        h0 = B.anslin_entropy_bits(counts[0])
        h1 = B.anslin_entropy_bits(counts[1][:16] if packed4 else counts[1])
        bpw = h0 + h1 if fmt == B.FMT_BF16 else (h0 / 2 if packed4 else h0)
        layers.append(dict(n_weights=n * (2 if packed4 else 1), counts=counts, h_coded=h0, h_side=h1, bits_per_weight=bpw))
    model = B.anslin_entropy_weighted([l["bits_per_weight"] for l in layers], [l["n_weights"] for l in layers])
    return dict(layers=layers, model_bits_per_weight=model)
