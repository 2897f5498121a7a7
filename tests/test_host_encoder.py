"""CPU tests of the product's host side through the C ABI: symbol export, anslin_encode_host vs the
oracle (cross-decode both ways), size accounting, validation in anslin_open.  No GPU calls."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import container as oc
from paper_2606_15789_b200 import binding as B
from paper_2606_15789_b200 import build as libbuild
from paper_2606_15789_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    libbuild.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "anslin.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(anslin_[a-z_0-9]+)\s*\(", hdr))
    assert names == set(B.EXPORTS)
    L = ctypes.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(L, n), n
    assert B.lib().anslin_status_string(4) == b"corrupt container"


def _cases():
    wf = inputs.weights_f32(256, 512, seed=31, jitter=True)
    yield "bf16", oc.FMT_BF16, inputs.f32_to_bf16_bits(wf), 512, dict(tile_k=64)
    yield "bf16-payload", oc.FMT_BF16, inputs.f32_to_bf16_bits(wf), 512, dict(tile_k=64, flags=1)
    yield "bf16-tile128", oc.FMT_BF16, inputs.f32_to_bf16_bits(wf), 512, dict(tile_k=128, flags=1)
    yield "bf16-32x256", oc.FMT_BF16, inputs.f32_to_bf16_bits(wf), 512, dict(tile_k=256, flags=1, tile_n=32)
    yield "bf16-32x64", oc.FMT_BF16, inputs.f32_to_bf16_bits(wf), 512, dict(tile_k=64, tile_n=32)
    yield "bf16-32x256-lanes", oc.FMT_BF16, inputs.f32_to_bf16_bits(wf), 512, dict(tile_k=256, flags=3, tile_n=32)
    yield "bf16-32x512-lanes", oc.FMT_BF16, inputs.f32_to_bf16_bits(wf), 512, dict(tile_k=512, flags=2, tile_n=32)
    q8, s8 = inputs.quant_sq8_weights(wf)
    yield "int8", oc.FMT_INT8, q8, 512, dict(tile_k=256, scales=s8)
    f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(128, 512, seed=32, std=0.015, outliers=False))
    yield "fp8", oc.FMT_FP8_E4M3, f8, 512, dict(tile_k=128, w_scale=sc)
    p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(128, 512, seed=33, outliers=False), 128)
    yield "int4", oc.FMT_INT4_AWQ, p4, 512, dict(tile_k=256, scales=s4, zeros=z4, group_size=128)
    yield "int8-32x256", oc.FMT_INT8, q8, 512, dict(tile_k=256, scales=s8, tile_n=32)
    yield "fp8-32x512", oc.FMT_FP8_E4M3, f8, 512, dict(tile_k=512, w_scale=sc, tile_n=32)
    yield "int4-32x512", oc.FMT_INT4_AWQ, p4, 512, dict(tile_k=512, scales=s4, zeros=z4, group_size=128, tile_n=32)
    yield "int8-32x512-lanes", oc.FMT_INT8, q8, 512, dict(tile_k=512, scales=s8, tile_n=32, flags=2)
    yield "fp8-32x256-lanes", oc.FMT_FP8_E4M3, f8, 512, dict(tile_k=256, w_scale=sc, tile_n=32, flags=2)
    yield "int4-32x512-lanes", oc.FMT_INT4_AWQ, p4, 512, dict(tile_k=512, scales=s4, zeros=z4, group_size=128, tile_n=32, flags=2)
    f5, sc5 = inputs.quant_fp8_e5m2_weights(inputs.weights_f32(128, 512, seed=34, std=0.015, outliers=False))
    yield "e5m2", oc.FMT_FP8_E5M2, f5, 512, dict(tile_k=256, w_scale=sc5)
    wp = inputs.f32_to_bf16_bits(wf).copy()
    wp[3, 5], wp[200, 300], wp[200, 301], wp[31, 511], wp[31, 510] = 0x0001, 0x7F7F, 0x0080, 0x0003, 0x7F00   # rare exponents: escapes
    yield "pair4-32x256-lanes-payload", oc.FMT_BF16_PAIR4, wp, 512, dict(tile_k=256, flags=3, tile_n=32)
    yield "pair4-32x512-lanes", oc.FMT_BF16_PAIR4, wp, 512, dict(tile_k=512, flags=2, tile_n=32)
    f4, sc4 = inputs.quant_fp4_weights(inputs.weights_f32(128, 512, seed=35, outliers=False))
    yield "fp4", oc.FMT_FP4_E2M1, f4, 512, dict(tile_k=256, w_scale=sc4)
    yield "fp4-32x512-lanes", oc.FMT_FP4_E2M1, f4, 512, dict(tile_k=512, w_scale=sc4, tile_n=32, flags=2)
    yield "e5m2-32x512-lanes", oc.FMT_FP8_E5M2, f5, 512, dict(tile_k=512, w_scale=sc5, tile_n=32, flags=2)


@pytest.mark.parametrize("name,fmt,w,k_in,kw", list(_cases()), ids=[c[0] for c in _cases()])
def test_cross_decode_and_stats(name, fmt, w, k_in, kw):
    n_out = w.shape[0]
    buf, st = B.anslin_encode_host(fmt, w, n_out, k_in, **kw)
    # the oracle decodes the library's container bit-exactly (P:l.26 strict losslessness)
    h, w2, side = oc.decode(buf)
    assert np.array_equal(w2.view(np.uint8), np.ascontiguousarray(w).view(np.uint8))
    if "scales" in kw:
        assert np.array_equal(side["scales"], kw["scales"])
    if "zeros" in kw:
        assert np.array_equal(side["zeros"], kw["zeros"])
    # the library accepts the oracle's container (header-only open; no device pointer)
    obuf, ost = oc.encode(fmt, w, k_in, **kw)
    hw = B.Weight(obuf, None)
    assert (hw.desc.n_out, hw.desc.k_in, hw.desc.tile_k, hw.desc.flags, hw.desc.tile_n) == \
        (n_out, k_in, kw["tile_k"], kw.get("flags", 0), kw.get("tile_n", 128))
    hw.close()
    B.Weight(buf, None).close()
    # both encoders are legal rANS coders over (possibly different) legal tables: sizes agree closely
    assert st["total_bytes"] == buf.size
    assert abs(st["bits_per_weight"] - ost["bits_per_weight"]) < 0.01
    assert st["entropy_bits_per_symbol"] == pytest.approx(ost["entropy_bits_per_symbol"], abs=1e-9)
    assert st["xent_bits_per_symbol"] >= st["entropy_bits_per_symbol"]
    wps = oc.WEIGHTS_PER_SYMBOL[fmt]
    assert st["bits_per_weight"] >= (st["entropy_bits_per_symbol"] + st["raw_entropy_bits_per_symbol"]) / wps
    total_bits = (st["payload_bits"] + st["state_bits"] + st["pad_bits"] + st["raw_bits"] + st["side_bits"])
    assert total_bits <= 8 * buf.size <= total_bits + st["offset_table_bits"] + st["freq_table_bits"] + 8 * (128 + 5 * 16 + 4096)


def test_entropy_functions_closed_forms_and_oracle():
    """anslin_entropy_bits / anslin_entropy_weighted (P:l.70, l.74): closed forms, and the oracle's own entropy of the
    same histogram (computed by the oracle's C routine behind container stats)."""
    assert B.anslin_entropy_bits(np.full(256, 7)) == pytest.approx(8.0, abs=1e-12)
    assert B.anslin_entropy_bits([5, 5]) == pytest.approx(1.0, abs=1e-12)
    assert B.anslin_entropy_bits([3, 1]) == pytest.approx(2.0 - 0.75 * np.log2(3.0), abs=1e-12)
    assert B.anslin_entropy_bits([0, 9, 0]) == 0.0 and B.anslin_entropy_bits(np.zeros(256)) == 0.0
    assert B.anslin_entropy_weighted([2.0, 4.0], [1, 3]) == pytest.approx(3.5, abs=1e-12)
    assert B.anslin_entropy_weighted([2.0], [0]) == 0.0
    w, _ = inputs.config1()
    _, ost = oc.encode(oc.FMT_BF16, w, 1024, tile_k=64)
    coded, raw = oc.symbolise(oc.FMT_BF16, w)
    assert B.anslin_entropy_bits(np.bincount(coded.ravel(), minlength=256)) == pytest.approx(ost["entropy_bits_per_symbol"], abs=1e-9)
    h = B.anslin_entropy_bits(np.bincount(coded.ravel(), minlength=256)) + B.anslin_entropy_bits(np.bincount(raw.ravel(), minlength=256))
    assert h == pytest.approx(ost["h_sym_bits_per_weight"], abs=1e-9)


def test_config1_gap_through_the_abi():
    """BASELINE target: bits/weight within 0.1 of the empirical entropy on config 1."""
    w, _ = inputs.config1()
    _, st = B.anslin_encode_host(B.FMT_BF16, w, 1024, 1024, tile_k=64, flags=B.FLAG_STATE_PAYLOAD)
    gap = st["bits_per_weight"] - (st["entropy_bits_per_symbol"] + st["raw_entropy_bits_per_symbol"])
    assert 0.0 <= gap <= 0.1


def test_unsupported_and_invalid_arguments():
    w = np.zeros((128, 64), dtype=np.uint16)
    with pytest.raises(B.AnslinError):
        B.anslin_encode_host(B.FMT_BF16, w, 100, 64)           # n_out not a multiple of 128
    with pytest.raises(B.AnslinError):
        B.anslin_encode_host(B.FMT_BF16, w, 128, 96)           # k_in not a multiple of tile_k
    with pytest.raises(B.AnslinError):
        B.anslin_encode_host(B.FMT_INT8, w, 128, 256, flags=1)  # payload flag is bf16-only
    d = B.Desc(B.FMT_INT8, 128, 256, 0, 0, 0, 1.0, 0)
    out = np.zeros(B.lib().anslin_encode_bound(ctypes.byref(d)), dtype=np.uint8)
    n = ctypes.c_size_t(0)
    rc = B.lib().anslin_encode_host(ctypes.byref(d), out.ctypes.data, None, None, out.ctypes.data, out.size, ctypes.byref(n), None)
    assert rc == 1                                              # int8 without scales: INVALID_ARG
    wq = np.zeros((128, 256), dtype=np.int8)
    sc = np.ones(128, dtype=np.float16)
    rc = B.lib().anslin_encode_host(ctypes.byref(d), wq.ctypes.data, sc.ctypes.data, None, out.ctypes.data, 64, ctypes.byref(n), None)
    assert rc == 3 and n.value > 64                             # BUFFER_TOO_SMALL reports the needed size


def test_open_rejects_corrupt_containers():
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(128, 128, seed=34))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, 128, 128, tile_k=64)
    h = oc.Header.unpack(buf)

    def status(b):
        out = ctypes.c_void_p()
        rc = B.lib().anslin_open(b.ctypes.data, b.size, None, ctypes.byref(out))
        if rc == 0:
            B.lib().anslin_close(out)
        return rc

    assert status(buf) == 0
    bad = buf.copy(); bad[0] ^= 1
    assert status(bad) == 4                                     # magic
    bad = buf.copy(); bad[h.off_freq] ^= 1
    assert status(bad) == 4                                     # table no longer sums to 4096
    bad = buf.copy(); bad[h.off_offsets + 4:h.off_offsets + 8] = 255
    assert status(bad) == 4                                     # tile offset out of range
    bad = buf.copy(); bad[12:16] = np.frombuffer(np.uint32(256).tobytes(), dtype=np.uint8)
    assert status(bad) == 4                                     # n_out inconsistent with n_tiles
    assert status(buf[:64].copy()) == 1                         # shorter than a header: INVALID_ARG


def test_open_checks_lane_stream_segment_tables():
    """the per-segment tables of a lane-stream record (u16 base, u16 total, 16 x u8 delta) become shared-memory
    cursors in the kernels, so anslin_open checks them whenever the host copy includes the records section."""
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(128, 512, seed=36, jitter=True))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, 128, 512, tile_k=256, flags=3, tile_n=32)
    h = oc.Header.unpack(buf)
    assert h.flags & 2

    def status(b, nbytes=None):
        out = ctypes.c_void_p()
        rc = B.lib().anslin_open(b.ctypes.data, b.size if nbytes is None else nbytes, None, ctypes.byref(out))
        if rc == 0:
            B.lib().anslin_close(out)
        return rc

    assert status(buf) == 0
    table = h.off_records + 128                    # first tile: 32 states, then the segment table
    for off, what in ((table, "base"), (table + 2, "total"), (table + 4, "delta[0]"), (table + 19, "delta[15]")):
        bad = buf.copy(); bad[off] ^= 0x40
        assert status(bad) == 4, what
    # the tables of a later tile are looked at as well
    offs = np.frombuffer(buf[h.off_offsets:h.off_offsets + 4 * (h.n_tiles + 1)].tobytes(), dtype=np.uint32)
    bad = buf.copy(); bad[h.off_records + 16 * int(offs[5]) + 128 + 7] ^= 0x20
    assert status(bad) == 4
    # a host copy that stops before the records (header + tables only) cannot be checked that far: accepted
    assert status(buf, int(h.off_records)) == 0


def test_gemm_entry_points_fail_loudly_without_a_device():
    """No CPU fallback: on a box without a GPU the device entry points return an error status."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(128, 128, seed=35))
    buf, _ = B.anslin_encode_host(B.FMT_BF16, w, 128, 128)
    hw = B.Weight(buf, None)
    with pytest.raises(B.AnslinError):
        B.anslin_decode(hw, 0, 0)
    with pytest.raises(B.AnslinError):
        B.anslin_gemm(hw, 16, B.DT_BF16, 128, 1, None, 16, 128, 16, 1 << 20)
    hw.close()


def test_widened_calls_validate_their_arguments_without_a_device():
    """The calls added for SURVEY 8(f) reject bad arguments before touching CUDA (so these checks run on any host)."""
    L = B.lib()
    ok = B.Desc(B.FMT_BF16, 256, 1024, 256, 0, B.FLAG_LANE_STREAMS | B.FLAG_STATE_PAYLOAD, 1.0, 32)
    assert L.anslin_encode_device_head_bytes(ctypes.byref(ok)) == 128 + 512 + 4 * (2 * 4 * 4 + 1) + 12    # header, table, offsets (aligned)
    assert L.anslin_encode_device_workspace_bytes(ctypes.byref(ok)) > 0
    for bad in (B.Desc(B.FMT_BF16, 256, 1024, 256, 0, B.FLAG_STATE_PAYLOAD, 1.0, 32),          # interleaved words: host encoder only
                B.Desc(B.FMT_BF16, 256, 1024, 256, 0, B.FLAG_LANE_STREAMS, 1.0, 128),          # 128-row tiles
                B.Desc(B.FMT_BF16, 256, 1024, 64, 0, B.FLAG_LANE_STREAMS, 1.0, 32),            # less than one segment per tile
                B.Desc(B.FMT_BF16_PAIR4, 256, 1024, 256, 0, B.FLAG_LANE_STREAMS, 1.0, 32),     # pair variant: host encoder only
                B.Desc(B.FMT_INT8, 256, 1024, 256, 0, B.FLAG_LANE_STREAMS | B.FLAG_STATE_PAYLOAD, 1.0, 32)):
        assert L.anslin_encode_device_head_bytes(ctypes.byref(bad)) == 0
        assert L.anslin_encode_device_workspace_bytes(ctypes.byref(bad)) == 0
    n = ctypes.c_size_t(0)
    assert L.anslin_encode_device(ctypes.byref(ok), None, None, None, None, 0, None, 0, None, 0, ctypes.byref(n), None) == 1   # INVALID_ARG
    assert L.anslin_histogram(B.FMT_BF16, None, 16, None, None) == 1
    buf = np.zeros(64, dtype=np.uint8)
    assert L.anslin_histogram(B.FMT_BF16, ctypes.c_void_p(buf.ctypes.data + 1), 16, ctypes.c_void_p(buf.ctypes.data), None) == 1   # misaligned
    assert L.anslin_histogram(99, ctypes.c_void_p(buf.ctypes.data), 16, ctypes.c_void_p(buf.ctypes.data), None) in (1, 2)
    with pytest.raises(B.AnslinError):
        B.anslin_encode_host(B.FMT_BF16_PAIR4, np.zeros((128, 256), np.uint16), 128, 256, tile_k=256, flags=0, tile_n=32)   # needs lane streams
    with pytest.raises(B.AnslinError):
        B.anslin_encode_host(B.FMT_BF16_PAIR4, np.zeros((128, 256), np.uint16), 128, 256, tile_k=256, flags=2, tile_n=128)
