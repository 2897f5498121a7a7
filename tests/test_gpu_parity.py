"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element.

Bars (BASELINE.json north_star): decoded weights bit-exact; GEMM max|d| <= 1e-2 * sum_k|x*w| per
element and relative Frobenius error <= 1e-3 (fp32 accumulate vs float64 oracle).
"""
import numpy as np
import pytest

from oracle import container as oc, gemm as og
from paper_2606_15789_b200 import binding as B
from paper_2606_15789_b200 import build as libbuild
from paper_2606_15789_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    libbuild.build()


def _rt():
    from paper_2606_15789_b200 import runtime
    return runtime


def check_gemm(y_gpu, y_ref, a_ref):
    y = y_gpu.astype(np.float64)
    assert np.all(np.isfinite(y))
    err = np.abs(y - y_ref)
    assert np.all(err <= 1e-2 * a_ref + 1e-30), "per-element bound: worst ratio %g" % float(np.max(err / (a_ref + 1e-30)))
    fro = np.linalg.norm(y - y_ref) / max(np.linalg.norm(y_ref), 1e-30)
    assert fro <= 1e-3, "relative Frobenius error %g" % fro


# ------------------------------------------------------------------ decode (a4-a7, a11)
def _decode_cases():
    wf = inputs.weights_f32(384, 640, seed=41, jitter=True)
    yield "bf16-t64", B.FMT_BF16, inputs.f32_to_bf16_bits(wf), 640, dict(tile_k=64)
    yield "bf16-t64-payload", B.FMT_BF16, inputs.f32_to_bf16_bits(wf), 640, dict(tile_k=64, flags=1)
    yield "bf16-t128-payload", B.FMT_BF16, inputs.f32_to_bf16_bits(wf), 640, dict(tile_k=128, flags=1)
    wf2 = inputs.weights_f32(256, 768, seed=42, jitter=True)
    q8, s8 = inputs.quant_sq8_weights(wf2)
    yield "int8", B.FMT_INT8, q8, 768, dict(tile_k=256, scales=s8)
    f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(256, 768, seed=43, std=0.015, outliers=False))
    yield "fp8", B.FMT_FP8_E4M3, f8, 768, dict(tile_k=128, w_scale=sc)
    p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(256, 768, seed=44, outliers=False), 128)
    yield "int4", B.FMT_INT4_AWQ, p4, 768, dict(tile_k=256, scales=s4, zeros=z4, group_size=128)
    yield "bf16-constant", B.FMT_BF16, np.full((128, 64), 0xBF80, dtype=np.uint16), 64, dict(tile_k=64)
    # 32-row tiles (four per MMA stripe), two tiles interleaved per warp
    yield "bf16-32x128-payload", B.FMT_BF16, inputs.f32_to_bf16_bits(wf), 640, dict(tile_k=128, flags=1, tile_n=32)
    yield "bf16-32x64", B.FMT_BF16, inputs.f32_to_bf16_bits(wf), 640, dict(tile_k=64, tile_n=32)
    yield "int8-32x256", B.FMT_INT8, q8, 768, dict(tile_k=256, scales=s8, tile_n=32)
    yield "fp8-32x384", B.FMT_FP8_E4M3, f8, 768, dict(tile_k=384, w_scale=sc, tile_n=32)
    yield "int4-32x256", B.FMT_INT4_AWQ, p4, 768, dict(tile_k=256, scales=s4, zeros=z4, group_size=128, tile_n=32)
    yield "bf16-constant-32", B.FMT_BF16, np.full((128, 64), 0xBF80, dtype=np.uint16), 64, dict(tile_k=64, tile_n=32)
    # lane-stream layout (every lane its own word stream, segments of 256 steps)
    wl = inputs.f32_to_bf16_bits(inputs.weights_f32(384, 1024, seed=45, jitter=True))
    yield "bf16-32x256-lanes-payload", B.FMT_BF16, wl, 1024, dict(tile_k=256, flags=3, tile_n=32)
    yield "bf16-32x512-lanes", B.FMT_BF16, wl, 1024, dict(tile_k=512, flags=2, tile_n=32)
    yield "int8-32x256-lanes", B.FMT_INT8, q8, 768, dict(tile_k=256, scales=s8, tile_n=32, flags=2)
    yield "fp8-32x768-lanes", B.FMT_FP8_E4M3, f8, 768, dict(tile_k=768, w_scale=sc, tile_n=32, flags=2)
    p4l, s4l, z4l = inputs.quant_awq4_weights(inputs.weights_f32(256, 1024, seed=46, outliers=False), 128)
    yield "int4-32x512-lanes", B.FMT_INT4_AWQ, p4l, 1024, dict(tile_k=512, scales=s4l, zeros=z4l, group_size=128, tile_n=32, flags=2)
    f5, sc5 = inputs.quant_fp8_e5m2_weights(inputs.weights_f32(256, 768, seed=47, std=0.015, outliers=False))
    yield "e5m2", B.FMT_FP8_E5M2, f5, 768, dict(tile_k=256, w_scale=sc5)
    yield "e5m2-32x768-lanes", B.FMT_FP8_E5M2, f5, 768, dict(tile_k=768, w_scale=sc5, tile_n=32, flags=2)
    f4, sc4 = inputs.quant_fp4_weights(inputs.weights_f32(256, 1024, seed=48, outliers=False))
    yield "fp4", B.FMT_FP4_E2M1, f4, 1024, dict(tile_k=256, w_scale=sc4)
    yield "fp4-32x256", B.FMT_FP4_E2M1, f4, 1024, dict(tile_k=256, w_scale=sc4, tile_n=32)
    yield "fp4-32x1024-lanes", B.FMT_FP4_E2M1, f4, 1024, dict(tile_k=1024, w_scale=sc4, tile_n=32, flags=2)
    wpair = wl.copy()
    wpair[3, 5], wpair[200, 300], wpair[200, 301], wpair[31, 1023], wpair[31, 1022], wpair[64, 255] = 0x0001, 0x7F7F, 0x0080, 0x0003, 0x7F00, 0xFF80
    yield "pair4-32x256-payload", B.FMT_BF16_PAIR4, wpair, 1024, dict(tile_k=256, flags=3, tile_n=32)
    yield "pair4-32x512", B.FMT_BF16_PAIR4, wpair, 1024, dict(tile_k=512, flags=2, tile_n=32)
    yield "pair4-constant", B.FMT_BF16_PAIR4, np.full((128, 256), 0xBF80, dtype=np.uint16), 256, dict(tile_k=256, tile_n=32, flags=3)
    yield "bf16-constant-lanes", B.FMT_BF16, np.full((128, 256), 0xBF80, dtype=np.uint16), 256, dict(tile_k=256, tile_n=32, flags=2)


@pytest.mark.parametrize("name,fmt,w,k_in,kw", list(_decode_cases()), ids=[c[0] for c in _decode_cases()])
@pytest.mark.parametrize("encoder", ["library", "oracle"])
def test_decode_bit_exact(name, fmt, w, k_in, kw, encoder):
    """decode(encode(W)) == W bit for bit (P:l.26, l.46, l.486), for containers from both encoders."""
    if encoder == "library":
        buf, _ = B.anslin_encode_host(fmt, w, w.shape[0], k_in, **kw)
    else:
        buf, _ = oc.encode(fmt, w, k_in, **kw)
    dw = _rt().DeviceWeight(buf)
    out = dw.decode().cpu().numpy()
    assert np.array_equal(out.view(np.uint8).reshape(w.shape[0], -1), np.ascontiguousarray(w).view(np.uint8).reshape(w.shape[0], -1))
    dw.close()


def test_decode_config1_full():
    w, _ = inputs.config1()
    for flags in (0, 1):
        buf, _ = B.anslin_encode_host(B.FMT_BF16, w, 1024, 1024, tile_k=64, flags=flags)
        dw = _rt().DeviceWeight(buf)
        assert np.array_equal(dw.decode().cpu().numpy().view(np.uint16), w)
        dw.close()


# ------------------------------------------------------------------ fused GEMM (a4-a10)
# (tile_n, bf16 tile_k, layout flag): BASELINE config 1's 128 x 64, 32-row tiles, and 32-row tiles with lane streams (bench.py)
TILES = [(128, 64, 0), (32, 256, 0), (32, 256, 2)]
TILE_IDS = ["128x64", "32x256", "32x256-lanes"]


@pytest.mark.parametrize("m", [1, 8, 16, 47, 75])
@pytest.mark.parametrize("flags", [0, 1])
@pytest.mark.parametrize("tile", TILES, ids=TILE_IDS)
def test_gemm_bf16(m, flags, tile):
    rt = _rt()
    n, k = 640, 1024      # 5 stripes x 16 (4) k-tiles: spans several CTAs and split-K segments
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=51, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=52))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=tile[1], flags=flags | tile[2], tile_n=tile[0])
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    y_ref, a_ref = og.gemm_bf16(x, w)
    check_gemm(y, y_ref, a_ref)
    dw.close()


@pytest.mark.parametrize("m", [1, 16, 75])
@pytest.mark.parametrize("tk,flags", [(256, 3), (512, 2)])
def test_gemm_bf16_pair_variant(m, tk, flags):
    """S: 8(f) NEXT-5: two K-adjacent bf16 exponents per rANS step (4-bit codes, escapes as in-stream literals);
    the GEMM sees exactly the original weights."""
    rt = _rt()
    n, k = 640, 1024
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=59, jitter=True)).copy()
    w[0, 0], w[639, 1023], w[300, 511], w[300, 512] = 0x0001, 0x5F7F, 0x0080, 0x8003    # rare exponents -> escapes (finite in fp32 sums)
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=60))
    buf, st = B.anslin_encode_host(B.FMT_BF16_PAIR4, w, n, k, tile_k=tk, flags=flags, tile_n=32)
    dw = rt.DeviceWeight(buf)
    assert np.array_equal(dw.decode().cpu().numpy().view(np.uint16), w)
    y = dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    check_gemm(y, *og.gemm_bf16(x, w))
    dw.close()


@pytest.mark.parametrize("tile", TILES, ids=TILE_IDS)
@pytest.mark.parametrize("m", [250, 256])
def test_gemm_bf16_max_batch_and_strided_buffers(m, tile):
    """Edge cases of the boundary: the largest single-block batch (m = 256, and 250 padded to 256 tensor-core
    columns), X and Y given as row-strided views (ldx > k_in, ldy > n_out): rows outside the views stay untouched."""
    rt = _rt()
    import torch
    n, k = 384, 1024
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=57, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=58))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=tile[1], flags=1 | tile[2], tile_n=tile[0])
    dw = rt.DeviceWeight(buf)
    xbig = torch.zeros((m, k + 64), dtype=torch.bfloat16, device="cuda")
    xbig[:, :k] = rt.x_to_device(B.FMT_BF16, x)
    ybig = torch.full((m, n + 32), -7.0, dtype=torch.float32, device="cuda")
    dw.gemm(xbig[:, :k], y=ybig[:, :n])
    y = ybig.cpu().numpy()
    check_gemm(y[:, :n], *og.gemm_bf16(x, w))
    assert np.all(y[:, n:] == -7.0)
    dw.close()


def test_gemm_multi_bf16_output():
    """anslin_gemm_multi_ex with bf16 Y: every element is the fp32 result rounded to nearest even, i.e. within one
    bf16 ulp of the float64 oracle's value rounded the same way (whole stripes and split-K stripes, odd row pitch)."""
    rt = _rt()
    import torch
    k, m = 2048, 37
    shapes = [640, 128]
    ws_, dws, refs = [], [], []
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=150))
    xd = rt.x_to_device(B.FMT_BF16, x)
    for i, n in enumerate(shapes):
        w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=151 + i, jitter=True))
        buf, _ = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=256, flags=3, tile_n=32)
        dws.append(rt.DeviceWeight(buf)); refs.append(og.gemm_bf16(x, w))
    ybig = [torch.full((m, n + 3), 7.0, dtype=torch.bfloat16, device="cuda") for n in shapes]      # odd pitch: scalar stores
    mg = rt.MultiGemm(dws, [xd, xd], None, [yb[:, :n] for yb, n in zip(ybig, shapes)])
    mg()
    mg32 = rt.MultiGemm(dws, [xd, xd])
    y32 = [t.cpu().numpy() for t in mg32()]
    for yb, n, (y_ref, a_ref), yf in zip(ybig, shapes, refs, y32):
        got = yb.float().cpu().numpy()
        assert np.all(got[:, n:] == 7.0)
        want = torch.from_numpy(yf).to(torch.bfloat16).float().numpy()          # RNE of the library's own fp32 result
        assert np.array_equal(got[:, :n], want)
        check_gemm(yf, y_ref, a_ref)
    for d in dws:
        d.close()


def test_gemm_replayed_from_a_cuda_graph():
    """A captured launch is replayed with its kernel parameters frozen, the split-K epoch among them: the stripe owner
    clears the flags it consumed, so every replay starts from "not stored" and sums this replay's partials."""
    rt = _rt()
    import torch
    n, k, m = 640, 2048, 33           # 8 k-tiles per stripe over many CTAs: every stripe is split
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=131, jitter=True))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=256, flags=3, tile_n=32)
    dw = rt.DeviceWeight(buf)
    xd = torch.zeros((m, k), dtype=torch.bfloat16, device="cuda")
    y = torch.zeros((m, n), dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        dw.gemm(xd, None, y)              # warm-up outside the capture: workspace allocation, function attributes
    torch.cuda.current_stream().wait_stream(side)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        dw.gemm(xd, None, y)
    for trial in range(3):
        x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=140 + trial))
        xd.copy_(rt.x_to_device(B.FMT_BF16, x))
        g.replay()
        torch.cuda.synchronize()
        check_gemm(y.cpu().numpy(), *og.gemm_bf16(x, w))
    dw.close()


@pytest.mark.parametrize("m", [257, 600, 2304])
def test_gemm_bf16_large_m(m):
    """S: §8(f) NEXT-1 (prefill-sized batches, P:l.392): m > 256 runs as blocks of 256 rows, 8 blocks per launch
    (2304 rows = two launches, the second with a single block); a ragged last block."""
    rt = _rt()
    n, k = 384, 1024
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=53, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=54))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=256, flags=3, tile_n=32)
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    check_gemm(y, *og.gemm_bf16(x, w))
    assert B.anslin_gemm_launches((m + 255) // 256) == (m + 2047) // 2048
    dw.close()


def test_gemm_int8_large_m_and_grouped_large_expert():
    rt = _rt()
    import torch
    n, k, m = 256, 1024, 300
    q, s = inputs.quant_sq8_weights(inputs.weights_f32(n, k, seed=63, jitter=True))
    xq, xs = inputs.quant_int8_acts(inputs.acts_f32(m, k, seed=64))
    buf, _ = B.anslin_encode_host(B.FMT_INT8, q, n, k, tile_k=256, scales=s)
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_INT8, xq), torch.from_numpy(xs).cuda()).cpu().numpy()
    y_ref, a_ref, _ = og.gemm_int8(xq, xs, q, s)       # per-token scales follow their rows into every block
    check_gemm(y, y_ref, a_ref)
    # grouped: expert 0 owns 280 rows (two problems), expert 1 none, expert 2 the remaining 20
    q2, s2 = inputs.quant_sq8_weights(inputs.weights_f32(n, k, seed=65, jitter=True))
    buf2, _ = B.anslin_encode_host(B.FMT_INT8, q2, n, k, tile_k=256, scales=s2)
    dw2, dw3 = rt.DeviceWeight(buf2), rt.DeviceWeight(buf)
    yg = rt.gemm_grouped([dw, dw3, dw2], [280, 0, 20], rt.x_to_device(B.FMT_INT8, xq), torch.from_numpy(xs).cuda()).cpu().numpy()
    check_gemm(yg[:280], y_ref[:280], a_ref[:280])
    y_ref2, a_ref2, _ = og.gemm_int8(xq[280:], xs[280:], q2, s2)
    check_gemm(yg[280:], y_ref2, a_ref2)
    for d in (dw, dw2, dw3):
        d.close()


@pytest.mark.parametrize("tile", TILES, ids=TILE_IDS)
def test_gemm_config1_and_unit_vector(tile):
    """BASELINE config 1 (W 1024x1024 bf16, X 8x1024) and the e_k special case: Y = column k of W exactly."""
    rt = _rt()
    w, x = inputs.config1()
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, 1024, 1024, tile_k=tile[1], flags=1 | tile[2], tile_n=tile[0])
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    check_gemm(y, *og.gemm_bf16(x, w))
    wf = og.bf16_bits_to_f64(w)
    for kk in (0, 7, 15, 16, 63, 64, 1000, 1023):
        e = np.zeros((1, 1024), dtype=np.float32); e[0, kk] = 1.0
        y = dw.gemm(rt.x_to_device(B.FMT_BF16, inputs.f32_to_bf16_bits(e))).cpu().numpy()
        assert np.array_equal(y[0].astype(np.float64), wf[:, kk]), "column %d" % kk
    dw.close()


LAYOUTS = [(128, 0), (32, 0), (32, 2)]      # (tile_n, layout flag)
LAYOUT_IDS = ["128", "32", "32-lanes"]


@pytest.mark.parametrize("lay", LAYOUTS, ids=LAYOUT_IDS)
@pytest.mark.parametrize("m", [1, 32, 75])
def test_gemm_int8(m, lay):
    tile_n, lflag = lay
    rt = _rt()
    import torch
    n, k = 384, 1536
    q, s = inputs.quant_sq8_weights(inputs.weights_f32(n, k, seed=61, jitter=True))
    xq, xs = inputs.quant_int8_acts(inputs.acts_f32(m, k, seed=62))
    buf, _ = B.anslin_encode_host(B.FMT_INT8, q, n, k, tile_k=256, scales=s, tile_n=tile_n, flags=lflag)
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_INT8, xq), torch.from_numpy(xs).cuda()).cpu().numpy()
    y_ref, a_ref, acc = og.gemm_int8(xq, xs, q, s)
    check_gemm(y, y_ref, a_ref)
    # integer sums are exact: undoing the (float) scales must round to the oracle's int64 sums
    back = np.rint(y.astype(np.float64) / (xs.astype(np.float64)[:, None] * s.astype(np.float64)[None, :]))
    small = np.abs(acc) < (1 << 22)
    assert np.array_equal(back[small], acc[small].astype(np.float64))
    dw.close()


@pytest.mark.parametrize("lay", LAYOUTS, ids=LAYOUT_IDS)
@pytest.mark.parametrize("m", [1, 20, 64])
def test_gemm_fp8(m, lay):
    tile_n, lflag = lay
    rt = _rt()
    import torch
    n, k = 256, 1536
    f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(n, k, seed=71, std=0.015, outliers=False))
    x8, xs = inputs.quant_fp8_acts(inputs.acts_f32(m, k, seed=72))
    buf, _ = B.anslin_encode_host(B.FMT_FP8_E4M3, f8, n, k, tile_k=256, w_scale=sc, tile_n=tile_n, flags=lflag)
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_FP8_E4M3, x8), torch.from_numpy(xs).cuda()).cpu().numpy()
    check_gemm(y, *og.gemm_fp8(x8, xs, f8, sc))
    dw.close()


@pytest.mark.parametrize("lay", LAYOUTS, ids=LAYOUT_IDS)
@pytest.mark.parametrize("m", [1, 16, 64])
def test_gemm_int4(m, lay):
    tile_n, lflag = lay
    rt = _rt()
    n, k = 256, 1024
    p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(n, k, seed=81, outliers=False), 128)
    x = inputs.acts_f32(m, k, seed=82).astype(np.float16)
    buf, _ = B.anslin_encode_host(B.FMT_INT4_AWQ, p4, n, k, tile_k=256 if tile_n == 128 else 512, scales=s4, zeros=z4,
                                  group_size=128, tile_n=tile_n, flags=lflag)
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_INT4_AWQ, x)).cpu().numpy()
    check_gemm(y, *og.gemm_int4(x, p4, s4, z4, 128))
    dw.close()


@pytest.mark.parametrize("lay", LAYOUTS, ids=LAYOUT_IDS)
def test_gemm_int4_plain_per_channel(lay):
    """S: §8(f) NEXT-2 "plain int4": symmetric per-channel int4 is the AWQ container with group_size = k_in and zero
    point 8; decode bit-exact, GEMM against (q - 8) * s[n] in float64."""
    tile_n, lflag = lay
    rt = _rt()
    n, k, m = 256, 1024, 24
    p4, s4, z4 = inputs.quant_int4_sym_weights(inputs.weights_f32(n, k, seed=83, outliers=False))
    x = inputs.acts_f32(m, k, seed=84).astype(np.float16)
    buf, st = B.anslin_encode_host(B.FMT_INT4_AWQ, p4, n, k, tile_k=256 if tile_n == 128 else 512, scales=s4, zeros=z4,
                                   group_size=k, tile_n=tile_n, flags=lflag)
    dw = rt.DeviceWeight(buf)
    assert np.array_equal(dw.decode().cpu().numpy(), p4)
    y = dw.gemm(rt.x_to_device(B.FMT_INT4_AWQ, x)).cpu().numpy()
    y_ref, a_ref = og.gemm_int4(x, p4, s4, z4, k)
    check_gemm(y, y_ref, a_ref)
    q = og.int4_unpack(p4).astype(np.float64) - 8.0
    assert np.allclose(y_ref, (x.astype(np.float64) @ q.T) * s4.astype(np.float64).T, rtol=1e-12, atol=1e-12)
    assert st["bits_per_weight"] < 4.0
    dw.close()


@pytest.mark.parametrize("lay", LAYOUTS, ids=LAYOUT_IDS)
@pytest.mark.parametrize("m", [1, 37])
@pytest.mark.parametrize("x_kind", ["e5m2", "e4m3"])
def test_gemm_fp8_e5m2(m, lay, x_kind):
    """NEXT-2 format fp8-E5M2 (P:l.80): same byte coder, tensor-core descriptor code e5m2 for W; X in either fp8 kind."""
    tile_n, lflag = lay
    rt = _rt()
    import torch
    n, k = 256, 1536
    f5, sc = inputs.quant_fp8_e5m2_weights(inputs.weights_f32(n, k, seed=73, std=0.015, outliers=False))
    xf = inputs.acts_f32(m, k, seed=74)
    x8, xs = inputs.quant_fp8_e5m2_acts(xf) if x_kind == "e5m2" else inputs.quant_fp8_acts(xf)
    buf, _ = B.anslin_encode_host(B.FMT_FP8_E5M2, f5, n, k, tile_k=256, w_scale=sc, tile_n=tile_n, flags=lflag)
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_FP8_E5M2, x8), torch.from_numpy(xs).cuda(),
                x_dtype=B.DT_FP8_E5M2 if x_kind == "e5m2" else B.DT_FP8_E4M3).cpu().numpy()
    check_gemm(y, *og.gemm_fp8(x8, xs, f5, sc, x_e5m2=x_kind == "e5m2", w_e5m2=True))
    dw.close()


@pytest.mark.parametrize("lay", LAYOUTS, ids=LAYOUT_IDS)
@pytest.mark.parametrize("m", [1, 37, 64])
def test_gemm_fp4(m, lay):
    """NEXT-2 format fp4-E2M1 (P:l.80): packed codes are the coded symbols; the decoder expands every code to the
    e4m3 byte of the same value, so the products are exact and only the fp32 accumulation rounds."""
    tile_n, lflag = lay
    rt = _rt()
    import torch
    n, k = 256, 2048
    p4, sc = inputs.quant_fp4_weights(inputs.weights_f32(n, k, seed=75, outliers=False))
    x8, xs = inputs.quant_fp8_acts(inputs.acts_f32(m, k, seed=76))
    buf, st = B.anslin_encode_host(B.FMT_FP4_E2M1, p4, n, k, tile_k=512, w_scale=sc, tile_n=tile_n, flags=lflag)
    assert st["bits_per_weight"] < 4.0
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_FP4_E2M1, x8), torch.from_numpy(xs).cuda()).cpu().numpy()
    check_gemm(y, *og.gemm_fp4(x8, xs, p4, sc))
    if m == 37:   # X in e5m2
        x5, xs5 = inputs.quant_fp8_e5m2_acts(inputs.acts_f32(m, k, seed=76))
        y = dw.gemm(rt.x_to_device(B.FMT_FP4_E2M1, x5), torch.from_numpy(xs5).cuda(), x_dtype=B.DT_FP8_E5M2).cpu().numpy()
        check_gemm(y, *og.gemm_fp4(x5, xs5, p4, sc, x_e5m2=True))
    dw.close()


@pytest.mark.parametrize("lay", LAYOUTS, ids=LAYOUT_IDS)
def test_gemm_grouped_fp8(lay):
    tile_n, lflag = lay
    """BASELINE config 5 in miniature: 8 experts, top-2 routing, rows sorted by expert."""
    rt = _rt()
    import torch
    n, k, E, tokens = 256, 768, 8, 20
    rows, tok = inputs.route_top2(tokens, E, seed=91)
    x8_tok, xs_tok = inputs.quant_fp8_acts(inputs.acts_f32(tokens, k, seed=92))
    x8, xs = x8_tok[tok], xs_tok[tok]
    experts, refs = [], []
    for e in range(E):
        f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(n, k, seed=100 + e, std=0.015, outliers=False))
        buf, _ = B.anslin_encode_host(B.FMT_FP8_E4M3, f8, n, k, tile_k=256, w_scale=sc, tile_n=tile_n, flags=lflag)
        experts.append(rt.DeviceWeight(buf))
        refs.append((f8, sc))
    y = rt.gemm_grouped(experts, rows, rt.x_to_device(B.FMT_FP8_E4M3, x8), torch.from_numpy(xs).cuda()).cpu().numpy()
    r0 = 0
    for e in range(E):
        r1 = r0 + int(rows[e])
        if r1 > r0:
            check_gemm(y[r0:r1], *og.gemm_fp8(x8[r0:r1], xs[r0:r1], refs[e][0], refs[e][1]))
        r0 = r1
    for d in experts:
        d.close()


def test_gemm_multi_qkv_shapes():
    """anslin_gemm_multi: three projections of different shapes that share one input, one launch."""
    rt = _rt()
    k, m = 1024, 47
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=95))
    xd = rt.x_to_device(B.FMT_BF16, x)
    ws, dws = [], []
    for i, n in enumerate((640, 128, 256)):
        w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=96 + i, jitter=True))
        buf, _ = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=256, flags=3, tile_n=32)
        ws.append(w); dws.append(rt.DeviceWeight(buf))
    mg = rt.MultiGemm(dws, [xd, xd, xd])
    ys = [y.cpu().numpy() for y in mg()]
    for w, y in zip(ws, ys):
        check_gemm(y, *og.gemm_bf16(x, w))
    ys2 = [y.cpu().numpy() for y in mg()]
    assert all(np.array_equal(a, b) for a, b in zip(ys, ys2)), "multi launch must be deterministic"
    for d in dws:
        d.close()


# ------------------------------------------------------------------ dense comparator
@pytest.mark.parametrize("m", [1, 16, 75])
def test_dense_gemm_bf16(m):
    rt = _rt()
    import torch
    n, k = 640, 1024
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=51, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=52))
    wd = torch.from_numpy(w.view(np.int16)).cuda()
    y = rt.dense_gemm(B.FMT_BF16, wd, rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    check_gemm(y, *og.gemm_bf16(x, w))


def test_dense_gemm_int8_fp8():
    rt = _rt()
    import torch
    n, k, m = 256, 1536, 32
    q, s = inputs.quant_sq8_weights(inputs.weights_f32(n, k, seed=61, jitter=True))
    xq, xs = inputs.quant_int8_acts(inputs.acts_f32(m, k, seed=62))
    y = rt.dense_gemm(B.FMT_INT8, torch.from_numpy(q).cuda(), rt.x_to_device(B.FMT_INT8, xq),
                      w_scale_vec=torch.from_numpy(s).cuda(), x_scale=torch.from_numpy(xs).cuda()).cpu().numpy()
    y_ref, a_ref, _ = og.gemm_int8(xq, xs, q, s)
    check_gemm(y, y_ref, a_ref)
    f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(n, k, seed=71, std=0.015, outliers=False))
    x8, xs8 = inputs.quant_fp8_acts(inputs.acts_f32(m, k, seed=72))
    y = rt.dense_gemm(B.FMT_FP8_E4M3, torch.from_numpy(f8).cuda(), rt.x_to_device(B.FMT_FP8_E4M3, x8), w_scale=sc,
                      x_scale=torch.from_numpy(xs8).cuda()).cpu().numpy()
    check_gemm(y, *og.gemm_fp8(x8, xs8, f8, sc))


def test_autotune_tile_picks_a_supported_geometry():
    """S: §8(f) NEXT-2 per-matrix tile-shape choice (P:l.167): every candidate must give the same Y within the
    GEMM tolerance; the winner is one of the rows, the size constraint is honoured."""
    rt = _rt()
    n, k, m = 512, 2048, 16
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=55, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=56))
    xd = rt.x_to_device(B.FMT_BF16, x)
    best, rows = rt.autotune_tile(B.FMT_BF16, w, n, k, m, xd, flags=B.FLAG_STATE_PAYLOAD, iters=5, max_gap_bits=0.05)
    assert len(rows) == len(rt.TILE_CANDIDATES) and best in rows
    assert best["bits_per_weight"] <= min(r["bits_per_weight"] for r in rows) + 0.05
    assert best["us"] == min(r["us"] for r in rows if r["bits_per_weight"] <= min(q["bits_per_weight"] for q in rows) + 0.05)
    y_ref, a_ref = og.gemm_bf16(x, w)
    for r in rows:
        dw = rt.DeviceWeight(r["container"])
        assert (dw.weight.desc.tile_n, dw.weight.desc.tile_k) == (r["tile_n"], r["tile_k"])
        check_gemm(dw.gemm(xd).cpu().numpy(), y_ref, a_ref)
        dw.close()


def test_histogram_and_entropy_study():
    """S: §8(f) NEXT-4 (P:l.64-78): device histograms are bit-exact against a bincount of the oracle's symbol planes,
    including a length that is not a multiple of the 16-byte vectors; model entropy = symbol-weighted mean."""
    rt = _rt()
    import torch
    wb = inputs.f32_to_bf16_bits(inputs.weights_f32(1031, 517, seed=111, jitter=True))        # odd element count
    coded, raw = oc.symbolise(oc.FMT_BF16, wb)
    f8, _ = inputs.quant_fp8_weights(inputs.weights_f32(640, 1027, seed=112, std=0.015, outliers=False))
    p4, _, _ = inputs.quant_awq4_weights(inputs.weights_f32(512, 2048, seed=113, outliers=False), 128)
    tb = torch.from_numpy(wb.view(np.int16)).cuda()
    st = rt.entropy_study(B.FMT_BF16, [tb, tb[:128].contiguous()])
    l0 = st["layers"][0]
    assert np.array_equal(l0["counts"][0], np.bincount(coded.ravel(), minlength=256).astype(np.uint64))
    assert np.array_equal(l0["counts"][1], np.bincount(raw.ravel(), minlength=256).astype(np.uint64))
    assert l0["n_weights"] == wb.size and int(l0["counts"][0].sum()) == wb.size
    _, ost = oc.encode(oc.FMT_BF16, np.ascontiguousarray(wb[:1024, :512]), 512, tile_k=64)
    sub = rt.entropy_study(B.FMT_BF16, [torch.from_numpy(np.ascontiguousarray(wb[:1024, :512]).view(np.int16)).cuda()])
    assert sub["layers"][0]["bits_per_weight"] == pytest.approx(ost["h_sym_bits_per_weight"], abs=1e-9)
    n0, n1 = st["layers"][0]["n_weights"], st["layers"][1]["n_weights"]
    ref = (n0 * st["layers"][0]["bits_per_weight"] + n1 * st["layers"][1]["bits_per_weight"]) / (n0 + n1)
    assert st["model_bits_per_weight"] == pytest.approx(ref, abs=1e-12)
    s8 = rt.entropy_study(B.FMT_FP8_E4M3, [torch.from_numpy(f8).cuda()])["layers"][0]
    assert np.array_equal(s8["counts"][0], np.bincount(f8.ravel(), minlength=256).astype(np.uint64)) and not s8["counts"][1].any()
    s4 = rt.entropy_study(B.FMT_INT4_AWQ, [torch.from_numpy(p4).cuda()])["layers"][0]
    assert np.array_equal(s4["counts"][0], np.bincount(p4.ravel(), minlength=256).astype(np.uint64))
    assert np.array_equal(s4["counts"][1][:16], np.bincount(og.int4_unpack(p4).ravel(), minlength=16).astype(np.uint64))
    assert s4["n_weights"] == 2 * p4.size and s4["bits_per_weight"] <= s4["h_side"] + 1e-12     # H(pair)/2 <= H(code)


def _device_encode_cases():
    wf = inputs.weights_f32(384, 1024, seed=121, jitter=True)
    yield "bf16-payload", B.FMT_BF16, inputs.f32_to_bf16_bits(wf), 1024, dict(tile_k=256, flags=3)
    yield "bf16-t512", B.FMT_BF16, inputs.f32_to_bf16_bits(wf), 1024, dict(tile_k=512, flags=2)
    q8, s8 = inputs.quant_sq8_weights(wf)
    yield "int8", B.FMT_INT8, q8, 1024, dict(tile_k=512, flags=2, scales=s8)
    f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(256, 1024, seed=122, std=0.015, outliers=False))
    yield "fp8-t1024", B.FMT_FP8_E4M3, f8, 1024, dict(tile_k=1024, flags=2, w_scale=sc)
    p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(256, 1024, seed=123, outliers=False), 128)
    yield "int4", B.FMT_INT4_AWQ, p4, 1024, dict(tile_k=512, flags=2, scales=s4, zeros=z4, group_size=128)
    yield "bf16-constant", B.FMT_BF16, np.full((128, 256), 0xBF80, dtype=np.uint16), 256, dict(tile_k=256, flags=3)


@pytest.mark.parametrize("name,fmt,w,k_in,kw", list(_device_encode_cases()), ids=[c[0] for c in _device_encode_cases()])
def test_encode_on_device(name, fmt, w, k_in, kw):
    """S: §8(f) NEXT-6 GPU-side encoder: the container it writes is decoded bit-exactly by the ORACLE and by
    anslin_decode, has the host encoder's table and (same table, same rANS arithmetic) the host encoder's size."""
    rt = _rt()
    import torch
    n_out = w.shape[0]
    wd = torch.from_numpy(np.ascontiguousarray(w).view(np.uint8).reshape(n_out, -1)).cuda()
    dw = rt.encode_on_device(fmt, wd, n_out, k_in, **kw)
    buf = dw.container_dev.cpu().numpy()
    h, w2, side = oc.decode(buf)
    assert np.array_equal(w2.view(np.uint8), np.ascontiguousarray(w).view(np.uint8))
    assert (h.tile_n, h.tile_k, h.flags) == (32, kw["tile_k"], kw["flags"])
    if "scales" in kw:
        assert np.array_equal(side["scales"], kw["scales"])
    assert np.array_equal(dw.decode().cpu().numpy().view(np.uint8).reshape(n_out, -1), np.ascontiguousarray(w).view(np.uint8).reshape(n_out, -1))
    hbuf, _ = B.anslin_encode_host(fmt, w, n_out, k_in, tile_n=32, **kw)
    assert buf.size == hbuf.size and np.array_equal(buf[:h.off_records], hbuf[:h.off_records])
    assert np.array_equal(buf, hbuf), "same table, same arithmetic, same layout: the two encoders agree byte for byte"
    dw.close()


def test_encode_on_device_then_gemm():
    rt = _rt()
    import torch
    n, k, m = 640, 1024, 20
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=124, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=125))
    dw = rt.encode_on_device(B.FMT_BF16, torch.from_numpy(w.view(np.int16)).cuda(), n, k, tile_k=256, flags=3)
    check_gemm(dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy(), *og.gemm_bf16(x, w))
    with pytest.raises(B.AnslinError):
        rt.encode_on_device(B.FMT_BF16, torch.from_numpy(w.view(np.int16)).cuda(), n, k, tile_k=64, flags=2)   # 64 steps: no whole segment
    dw.close()


# ------------------------------------------------------------------ full-size launch configuration
@pytest.mark.parametrize("tile", TILES, ids=TILE_IDS)
@pytest.mark.parametrize("name,n,k,m", [("gate", 13824, 5120, 75), ("down", 5120, 13824, 16), ("k", 1024, 5120, 1)])
def test_gemm_bf16_full_size_projection(name, n, k, m, tile):
    """BASELINE config 2 shapes in the launch configuration bench.py times (148 persistent CTAs,
    ~58 tiles per CTA, several ring laps and split-K segments per CTA): decode bit-exact on the
    full tensor, GEMM checked on all M rows x a seeded sample of 1024 output channels."""
    rt = _rt()
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=7, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=8))
    buf, st = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=tile[1], flags=1 | tile[2], tile_n=tile[0])
    assert st["bits_per_weight"] - st["entropy_bits_per_symbol"] - st["raw_entropy_bits_per_symbol"] <= 0.1
    dw = rt.DeviceWeight(buf)
    assert np.array_equal(dw.decode().cpu().numpy().view(np.uint16), w)
    y = dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    cols = np.sort(np.random.default_rng(9).choice(n, size=min(n, 1024), replace=False))
    y_ref, a_ref = og.gemm_bf16(x, w[cols])
    check_gemm(y[:, cols], y_ref, a_ref)
    y2 = dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    assert np.array_equal(y, y2), "split-K fix-up must be deterministic"
    dw.close()


def test_gemm_bf16_odd_k_tiles_pair_items():
    """An odd number of k-tiles per stripe on the tensor-memory kernel's PAIR work items (the last pair of a stripe has one
    tile; more tiles than teams, so the one-tile work items of small launches are not chosen): 4096 x 4864 bf16, 19 k-tiles
    of 256, M = 20, lane streams + payload; decode bit-exact, GEMM on sampled channels, run-to-run bit equality."""
    rt = _rt()
    n, k, m = 4096, 4864, 20
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=131, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=132))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=256, flags=3, tile_n=32)
    dw = rt.DeviceWeight(buf)
    assert np.array_equal(dw.decode().cpu().numpy().view(np.uint16), w)
    xd = rt.x_to_device(B.FMT_BF16, x)
    y = dw.gemm(xd).cpu().numpy()
    cols = np.sort(np.random.default_rng(133).choice(n, size=768, replace=False))
    check_gemm(y[:, cols], *og.gemm_bf16(x, w[cols]))
    assert np.array_equal(y, dw.gemm(xd).cpu().numpy())
    dw.close()


# ------------------------------------------------------------------ BASELINE configs 3-5 at full size
def _sample_cols(n, seed, count=512):
    return np.sort(np.random.default_rng(seed).choice(n, size=min(n, count), replace=False))


def test_pair_variant_and_device_encoder_full_size():
    """The two widened paths at a BASELINE config 2 shape (o: 5120 x 5120, M = 47) in the launch configuration
    bench.py times: the bf16 pair variant decodes bit-exactly and multiplies in tolerance, with its own size gap
    stated; the GPU-side encoder reproduces the host encoder's container byte for byte."""
    rt = _rt()
    import torch
    n, k, m = 5120, 5120, 47
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=17, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=18))
    buf, st = B.anslin_encode_host(B.FMT_BF16_PAIR4, w, n, k, tile_k=256, flags=3, tile_n=32)
    buf0, st0 = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=256, flags=3, tile_n=32)
    assert 0.0 < st["bits_per_weight"] - st0["bits_per_weight"] < 0.03
    dw = rt.DeviceWeight(buf)
    assert np.array_equal(dw.decode().cpu().numpy().view(np.uint16), w)
    cols = np.sort(np.random.default_rng(19).choice(n, size=1024, replace=False))
    y = dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    check_gemm(y[:, cols], *og.gemm_bf16(x, w[cols]))
    dw.close()
    de = rt.encode_on_device(B.FMT_BF16, torch.from_numpy(w.view(np.int16)).cuda(), n, k, tile_k=256, flags=3)
    assert np.array_equal(de.container_dev.cpu().numpy(), buf0)
    de.close()


@pytest.mark.parametrize("lay", [(128, 256, 0), (32, 1024, 2)], ids=["128x256", "32x1024-lanes"])
def test_config3_int8_full_size(lay):
    """BASELINE config 3: Qwen-14B gate projection 13824 x 5120 in SQ8-style int8, M = 75: decode bit-exact on the
    whole tensor, fused GEMM on all rows x sampled channels, integer sums exact, bits/weight within 0.1 of H."""
    rt = _rt()
    import torch
    n, k, m = 13824, 5120, 75
    q, s = inputs.quant_sq8_weights(inputs.weights_f32(n, k, seed=5, jitter=True))
    xq, xs = inputs.quant_int8_acts(inputs.acts_f32(m, k, seed=6))
    buf, st = B.anslin_encode_host(B.FMT_INT8, q, n, k, tile_k=lay[1], scales=s, tile_n=lay[0], flags=lay[2])
    assert 0.0 <= st["bits_per_weight"] - st["entropy_bits_per_symbol"] <= 0.1
    dw = rt.DeviceWeight(buf)
    assert np.array_equal(dw.decode().cpu().numpy().view(np.int8), q)
    y = dw.gemm(rt.x_to_device(B.FMT_INT8, xq), torch.from_numpy(xs).cuda()).cpu().numpy()
    cols = _sample_cols(n, 9)
    y_ref, a_ref, acc = og.gemm_int8(xq, xs, q[cols], s[cols])
    check_gemm(y[:, cols], y_ref, a_ref)
    back = np.rint(y[:, cols].astype(np.float64) / (xs.astype(np.float64)[:, None] * s[cols].astype(np.float64)[None, :]))
    small = np.abs(acc) < (1 << 22)
    assert np.array_equal(back[small], acc[small].astype(np.float64))
    dw.close()


@pytest.mark.parametrize("lay", [(128, 256, 0), (32, 1024, 2)], ids=["128x256", "32x1024-lanes"])
def test_config4_int4_full_size(lay):
    """BASELINE config 4: Llama-70B gate projection 28672 x 8192, AWQ-style int4 (group 128), fp16 X, M = 64."""
    rt = _rt()
    n, k, m = 28672, 8192, 64
    p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(n, k, seed=11, outliers=False), 128)
    x = inputs.acts_f32(m, k, seed=12).astype(np.float16)
    buf, st = B.anslin_encode_host(B.FMT_INT4_AWQ, p4, n, k, tile_k=lay[1], scales=s4, zeros=z4, group_size=128, tile_n=lay[0],
                                  flags=lay[2])
    assert 0.0 <= st["bits_per_weight"] - st["entropy_bits_per_symbol"] / 2 <= 0.1
    dw = rt.DeviceWeight(buf)
    assert np.array_equal(dw.decode().cpu().numpy(), p4)
    y = dw.gemm(rt.x_to_device(B.FMT_INT4_AWQ, x)).cpu().numpy()
    cols = _sample_cols(n, 13)
    check_gemm(y[:, cols], *og.gemm_int4(x, p4[cols], s4[cols], z4[cols], 128))
    dw.close()


@pytest.mark.parametrize("lay", [(128, 256, 0), (32, 1024, 2)], ids=["128x256", "32x1024-lanes"])
def test_config5_fp8_moe_full_size(lay):
    """BASELINE config 5: 8 Mixtral-8x22B-shaped experts (gate 16384 x 6144, e4m3), 95 tokens routed top-2:
    one grouped persistent launch over the active experts; every expert's rows checked on sampled channels."""
    rt = _rt()
    import torch
    n, k, E, tokens = 16384, 6144, 8, 95
    rows, tok = inputs.route_top2(tokens, E, seed=21)
    x8_tok, xs_tok = inputs.quant_fp8_acts(inputs.acts_f32(tokens, k, seed=22))
    x8, xs = x8_tok[tok], xs_tok[tok]
    experts, refs = [], []
    for e in range(E):
        f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(n, k, seed=30 + e, std=0.015, outliers=False))
        buf, st = B.anslin_encode_host(B.FMT_FP8_E4M3, f8, n, k, tile_k=lay[1], w_scale=sc, tile_n=lay[0], flags=lay[2])
        assert 0.0 <= st["bits_per_weight"] - st["entropy_bits_per_symbol"] <= 0.1
        experts.append(rt.DeviceWeight(buf))
        refs.append((f8, sc))
    assert np.array_equal(experts[3].decode().cpu().numpy(), refs[3][0])
    y = rt.gemm_grouped(experts, rows, rt.x_to_device(B.FMT_FP8_E4M3, x8), torch.from_numpy(xs).cuda()).cpu().numpy()
    r0 = 0
    for e in range(E):
        r1 = r0 + int(rows[e])
        if r1 > r0:
            cols = _sample_cols(n, 40 + e, 256)
            check_gemm(y[r0:r1][:, cols], *og.gemm_fp8(x8[r0:r1], xs[r0:r1], refs[e][0][cols], refs[e][1]))
        r0 = r1
    for d in experts:
        d.close()


# ------------------------------------------------------------------ the long-K `down` projections of configs 3-5
@pytest.mark.parametrize("m", [1, 75])
def test_config3_int8_down_long_k(m):
    """BASELINE config 3 `down`: 5120 x 13824 int8 (K = 13824: 54 k-tiles, the long accumulation), M in {1, 75}: fused GEMM on all
    rows x sampled channels inside both tolerances, integer sums exact."""
    rt = _rt()
    import torch
    n, k = 5120, 13824
    q, s = inputs.quant_sq8_weights(inputs.weights_f32(n, k, seed=61, jitter=True))
    xq, xs = inputs.quant_int8_acts(inputs.acts_f32(m, k, seed=62))
    buf, st = B.anslin_encode_host(B.FMT_INT8, q, n, k, tile_k=512, scales=s, tile_n=32, flags=2)
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_INT8, xq), torch.from_numpy(xs).cuda()).cpu().numpy()
    cols = _sample_cols(n, 63)
    y_ref, a_ref, acc = og.gemm_int8(xq, xs, q[cols], s[cols])
    check_gemm(y[:, cols], y_ref, a_ref)
    back = np.rint(y[:, cols].astype(np.float64) / (xs.astype(np.float64)[:, None] * s[cols].astype(np.float64)[None, :]))
    small = np.abs(acc) < (1 << 22)
    assert np.array_equal(back[small], acc[small].astype(np.float64))
    dw.close()


@pytest.mark.parametrize("m", [1, 64])
def test_config4_int4_down_long_k(m):
    """BASELINE config 4 `down`: 8192 x 28672 AWQ int4 (224 groups of 128 along K, fp16 dequantisation rounding accumulated over
    28672 terms), fp16 X, M in {1, 64}."""
    rt = _rt()
    n, k = 8192, 28672
    p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(n, k, seed=64, outliers=False), 128)
    x = inputs.acts_f32(m, k, seed=65).astype(np.float16)
    buf, st = B.anslin_encode_host(B.FMT_INT4_AWQ, p4, n, k, tile_k=1024, scales=s4, zeros=z4, group_size=128, tile_n=32, flags=2)
    assert 0.0 <= st["bits_per_weight"] - st["entropy_bits_per_symbol"] / 2 <= 0.1
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_INT4_AWQ, x)).cpu().numpy()
    cols = _sample_cols(n, 66)
    check_gemm(y[:, cols], *og.gemm_int4(x, p4[cols], s4[cols], z4[cols], 128))
    dw.close()


@pytest.mark.parametrize("tokens", [20, 95])
def test_config5_fp8_moe_down_long_k(tokens):
    """BASELINE config 5 `down`: 8 experts 6144 x 16384 e4m3 (K = 16384, the case SURVEY 7-8 flags for fp8 accumulation
    precision), `tokens` tokens routed top-2, one grouped launch; every active expert's rows on sampled channels."""
    rt = _rt()
    import torch
    n, k, E = 6144, 16384, 8
    rows, tok = inputs.route_top2(tokens, E, seed=71)
    x8_tok, xs_tok = inputs.quant_fp8_acts(inputs.acts_f32(tokens, k, seed=72))
    x8, xs = x8_tok[tok], xs_tok[tok]
    experts, refs = [], []
    for e in range(E):
        f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(n, k, seed=80 + e, std=0.015, outliers=False))
        buf, st = B.anslin_encode_host(B.FMT_FP8_E4M3, f8, n, k, tile_k=1024, w_scale=sc, tile_n=32, flags=2)
        experts.append(rt.DeviceWeight(buf))
        refs.append((f8, sc))
    y = rt.gemm_grouped(experts, rows, rt.x_to_device(B.FMT_FP8_E4M3, x8), torch.from_numpy(xs).cuda()).cpu().numpy()
    r0 = 0
    for e in range(E):
        r1 = r0 + int(rows[e])
        if r1 > r0:
            cols = _sample_cols(n, 90 + e, 256)
            check_gemm(y[r0:r1][:, cols], *og.gemm_fp8(x8[r0:r1], xs[r0:r1], refs[e][0][cols], refs[e][1]))
        r0 = r1
    for d in experts:
        d.close()


@pytest.mark.parametrize("name", ["q", "o"])
def test_config2_bf16_square_projection_m47(name):
    """BASELINE config 2 q / o: 5120 x 5120 plain bf16 at M = 47 (the paper's uncompressed max batch, P:l.378)."""
    rt = _rt()
    n = k = 5120
    m = 47
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=101 if name == "q" else 102, jitter=True))
    x = inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=103))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=256, flags=3, tile_n=32)
    dw = rt.DeviceWeight(buf)
    y = dw.gemm(rt.x_to_device(B.FMT_BF16, x)).cpu().numpy()
    cols = _sample_cols(n, 104, 1024)
    check_gemm(y[:, cols], *og.gemm_bf16(x, w[cols]))
    dw.close()


def test_bench_step_full_size():
    """Exactly the step bench.py times: the Qwen-14B-shaped bf16 layer at M = 75, 32 x 256 tiles, lane streams + payload, four
    persistent multi-problem launches (q+k+v, o, gate+up, down) whose problems share the SMs.  Every Y is checked against the
    float64 oracle on 512 sampled channels per projection, and a second run must reproduce every Y bit for bit."""
    rt = _rt()
    import torch
    m = 75
    layer = [(nm, n, k, inputs.f32_to_bf16_bits(inputs.weights_f32(n, k, seed=1 + i, jitter=True)))
             for i, (nm, n, k) in enumerate(inputs.QWEN14B_LAYER)]
    names = [t[0] for t in layer]
    dws = [rt.DeviceWeight(B.anslin_encode_host(B.FMT_BF16, w, n, k, tile_k=256, flags=3, tile_n=32)[0]) for (_, n, k, w) in layer]
    share = {"k": "q", "v": "q", "up": "gate"}
    xs_np = {nm: inputs.f32_to_bf16_bits(inputs.acts_f32(m, k, seed=500 + i)) for i, (nm, n, k, _) in enumerate(layer) if nm not in share}
    xs_dev = {nm: rt.x_to_device(B.FMT_BF16, x) for nm, x in xs_np.items()}
    groups = [["q", "k", "v"], ["o"], ["gate", "up"], ["down"]]
    calls = [rt.MultiGemm([dws[names.index(nm)] for nm in g], [xs_dev[share.get(nm, nm)] for nm in g]) for g in groups]
    first = None
    for rep in range(2):
        ys = {}
        for g, call in zip(groups, calls):
            for nm, y in zip(g, call()):
                ys[nm] = y
        torch.cuda.synchronize()
        got = {nm: y.cpu().numpy().copy() for nm, y in ys.items()}
        if first is None:
            first = got
        else:
            for nm in names:
                assert np.array_equal(first[nm], got[nm]), "run-to-run difference in " + nm
    for i, (nm, n, k, w) in enumerate(layer):
        cols = _sample_cols(n, 600 + i, 512)
        check_gemm(first[nm][:, cols], *og.gemm_bf16(xs_np[share.get(nm, nm)], w[cols]))
    for d in dws:
        d.close()
