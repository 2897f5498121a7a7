"""anslin_gemm_static: the fused decode-GEMM on the library's static device workspace (no allocation inside the call).

Collected last on purpose (the suite runs with pytest -x).  Checked against the existing path (anslin_gemm with a
caller-owned workspace: same kernel, same grid, same reduction order, so bit for bit) and against the float64 oracle
within the bars of tests/test_gpu_parity.py, on two calls in a row that share the static array.
"""
import numpy as np
import pytest

from oracle import gemm as og
from paper_2606_15789_b200 import binding as B
from paper_2606_15789_b200 import build as libbuild
from paper_2606_15789_b200 import inputs

pytestmark = pytest.mark.gpu


def _check_gemm(y_gpu, y_ref, a_ref):   # north_star bars, as in test_gpu_parity.check_gemm
    y = y_gpu.astype(np.float64)
    assert np.all(np.isfinite(y))
    err = np.abs(y - y_ref)
    assert np.all(err <= 1e-2 * a_ref + 1e-30), "per-element bound: worst ratio %g" % float(np.max(err / (a_ref + 1e-30)))
    fro = np.linalg.norm(y - y_ref) / max(np.linalg.norm(y_ref), 1e-30)
    assert fro <= 1e-3, "relative Frobenius error %g" % fro


def test_gemm_static_matches_gemm_on_two_calls_in_a_row():
    libbuild.build()
    import torch
    from paper_2606_15789_b200 import runtime as rt
    # call 1: bf16, lane streams, 32 x 256 tiles -> tensor-memory kernel, every stripe split over several teams (split-K
    # flags and partials in the static array); call 2: another matrix, shape, format and kernel (int8, 32 x 1024 tiles of a
    # short-and-wide matrix -> shared-memory operand design) on the same array, which still holds call 1's bytes
    n1, k1, m1 = 1024, 5120, 16
    w1 = inputs.f32_to_bf16_bits(inputs.weights_f32(n1, k1, seed=901, jitter=True))
    x1 = inputs.f32_to_bf16_bits(inputs.acts_f32(m1, k1, seed=902))
    d1 = rt.DeviceWeight(B.anslin_encode_host(B.FMT_BF16, w1, n1, k1, tile_k=256, flags=3, tile_n=32)[0])
    n2, k2, m2 = 768, 4096, 29
    q8, s8 = inputs.quant_sq8_weights(inputs.weights_f32(n2, k2, seed=903, jitter=True))
    xq, xs = inputs.quant_int8_acts(inputs.acts_f32(m2, k2, seed=904))
    d2 = rt.DeviceWeight(B.anslin_encode_host(B.FMT_INT8, q8, n2, k2, tile_k=1024, flags=2, tile_n=32, scales=s8)[0])
    x1d, x2d, xsd = rt.x_to_device(B.FMT_BF16, x1), rt.x_to_device(B.FMT_INT8, xq), torch.from_numpy(xs).cuda()
    ref1 = d1.gemm(x1d).cpu().numpy()
    ref2 = d2.gemm(x2d, xsd).cpu().numpy()
    y1 = torch.full((m1, n1), float("nan"), dtype=torch.float32, device="cuda")
    y2 = torch.full((m2, n2), float("nan"), dtype=torch.float32, device="cuda")
    for rep in range(2):   # two rounds of two calls in a row, no synchronisation in between: stream order is the only order
        d1.gemm_static(x1d, y=y1)
        d2.gemm_static(x2d, xsd, y=y2)
        torch.cuda.synchronize()
        got1, got2 = y1.cpu().numpy(), y2.cpu().numpy()
        assert np.array_equal(got1, ref1), "static workspace, call 1 of round %d differs from anslin_gemm" % rep
        assert np.array_equal(got2, ref2), "static workspace, call 2 of round %d differs from anslin_gemm" % rep
        y1.fill_(float("nan")); y2.fill_(float("nan"))
    _check_gemm(got1, *og.gemm_bf16(x1, w1))
    _check_gemm(got2, *og.gemm_int8(xq, xs, q8, s8)[:2])
    # beyond the array: refused with its own status, nothing enqueued
    big = torch.zeros((200, k1), dtype=torch.bfloat16, device="cuda")
    assert B.anslin_gemm_workspace_bytes(d1.weight, 200) > B.STATIC_WORKSPACE_BYTES
    with pytest.raises(B.AnslinError, match="static workspace"):
        d1.gemm_static(big)
    d1.close(); d2.close()
