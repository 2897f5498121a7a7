"""Pins for the oracle's container, symbolisation, metadata model and reference GEMM.  CPU only."""
import os

import numpy as np
import pytest

from oracle import codec, container as oc, gemm as og
from paper_2606_15789_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_table3_from_eq3():
    """Eq.3 (P:l.440) reproduces every printed value of Table III (P:l.456-466)."""
    for line in open(os.path.join(GOLD, "table3.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        rows, cols = int(t[1]), int(t[2])
        for (tr, tc), (kb, pct, eff) in (((32, 128), map(float, t[3:6])), ((64, 256), map(float, t[6:9]))):
            n_tiles = (rows // tr) * (cols // tc)
            meta = oc.metadata_bytes_eq3(n_tiles, 12)
            assert round(meta / 1024.0, 1) == pytest.approx(kb, abs=0.051)
            assert 100.0 * meta / (rows * cols * 2) == pytest.approx(pct, abs=0.0006)
            assert 16.0 * meta / (rows * cols * 2) == pytest.approx(eff, abs=0.00006)


def test_symbolise_bf16_is_a_bijection_on_all_65536_codes():
    bits = np.arange(65536, dtype=np.uint16).reshape(256, 256)
    coded, raw = oc.symbolise(oc.FMT_BF16, bits)
    assert np.array_equal(oc.desymbolise(oc.FMT_BF16, coded, raw), bits)
    # coded plane is the IEEE exponent field: check against frexp on the float value
    f = inputs.bf16_bits_to_f32(bits)
    normal = np.isfinite(f) & (np.abs(f) >= 2.0 ** -126)
    _, e = np.frexp(f[normal])
    assert np.array_equal(coded[normal].astype(np.int64), e + 126)
    assert np.array_equal(raw & 1, (bits >> 15).astype(np.uint8))


@pytest.mark.parametrize("fmt,tile_k,tile_n", [(oc.FMT_BF16, 64, 128), (oc.FMT_FP8_E4M3, 256, 128), (oc.FMT_INT8, 128, 128),
                                               (oc.FMT_INT4_AWQ, 256, 128), (oc.FMT_BF16, 256, 32), (oc.FMT_INT8, 256, 32),
                                               (oc.FMT_INT4_AWQ, 512, 32)])
def test_tile_order_is_a_permutation_with_chunk_structure(fmt, tile_k, tile_n):
    rows, cols = oc.tile_order(fmt, tile_k, tile_n)
    sym_cols = tile_k // oc.WEIGHTS_PER_SYMBOL[fmt]
    assert rows.size == tile_n * sym_cols
    if tile_n == 32:      # lane l simply walks row l in K order
        assert np.array_equal(rows.reshape(-1, 32), np.tile(np.arange(32), (sym_cols, 1)))
        assert np.array_equal(cols.reshape(-1, 32), np.tile(np.arange(sym_cols)[:, None], (1, 32)))
    assert np.unique(rows * sym_cols + cols).size == rows.size
    spc = oc.SPC[fmt]
    # a lane's spc consecutive steps are spc consecutive symbol columns of one row = one 16-byte operand chunk
    r = rows.reshape(-1, spc, 32)
    c = cols.reshape(-1, spc, 32)
    assert np.all(r == r[:, :1, :]) and np.all(np.diff(c, axis=1) == 1) and np.all(c[:, 0, :] % spc == 0)


def _roundtrip(fmt, w, k_in, **kw):
    buf, st = oc.encode(fmt, w, k_in, **kw)
    h, w2, side = oc.decode(buf)
    assert w2.shape == w.shape and np.array_equal(w2.view(np.uint8), np.ascontiguousarray(w).view(np.uint8))
    assert st["total_bytes"] == buf.size == h.total_bytes
    return buf, st, h, side


def test_roundtrip_bf16_config1_and_bits_per_weight_gate():
    """Strict losslessness (P:l.26, l.46, l.486) and the size bound (P:l.12: within 0.01-0.1 bit of
    the Shannon bound) on BASELINE config 1, with and without the initial-state payload (A4)."""
    w, _ = inputs.config1()
    _, st0, _, _ = _roundtrip(oc.FMT_BF16, w, 1024, tile_k=64, flags=0)
    _, st1, h1, _ = _roundtrip(oc.FMT_BF16, w, 1024, tile_k=64, flags=oc.FLAG_STATE_PAYLOAD)
    for st in (st0, st1):
        assert st["bits_per_weight"] >= st["h_sym_bits_per_weight"]
        assert st["xent_bits_per_symbol"] >= st["entropy_bits_per_symbol"]
    assert st1["bits_per_weight"] < st0["bits_per_weight"]
    assert st1["bits_per_weight"] - st1["h_sym_bits_per_weight"] <= 0.1
    assert 0.1 < st0["bits_per_weight"] - st0["h_sym_bits_per_weight"] <= 0.2     # P:l.366 "roughly 0.1-0.2 bits"
    # per-stream flush overhead in (16, 32] bits without payload
    ideal = st0["xent_bits_per_symbol"] * st0["n_weights"]
    per_stream = (st0["payload_bits"] + st0["state_bits"] - ideal) / (h1.n_tiles * 32)
    assert 16.0 < per_stream <= 32.0
    # metadata accounting: one 4-byte offset per tile (Eq.3's first term) + one sentinel
    assert st0["offset_table_bits"] == 32 * (h1.n_tiles + 1)
    # brute-force entropy of the symbol planes, independent of the oracle's C routine
    coded, raw = oc.symbolise(oc.FMT_BF16, w)
    H = 0.0
    for plane in (coded, raw):
        p = np.bincount(plane.ravel(), minlength=256) / plane.size
        H -= float(np.sum(p[p > 0] * np.log2(p[p > 0])))
    assert st0["h_sym_bits_per_weight"] == pytest.approx(H, abs=1e-9)


def test_roundtrip_int8_fp8_int4_small():
    wf = inputs.weights_f32(256, 512, seed=11, jitter=True)
    q8, s8 = inputs.quant_sq8_weights(wf)
    _, st, _, side = _roundtrip(oc.FMT_INT8, q8, 512, tile_k=256, scales=s8)
    assert np.array_equal(side["scales"], s8) and st["bits_per_weight"] >= st["h_sym_bits_per_weight"]
    f8, sc = inputs.quant_fp8_weights(inputs.weights_f32(128, 512, seed=12, std=0.015, outliers=False))
    _, st, h, _ = _roundtrip(oc.FMT_FP8_E4M3, f8, 512, tile_k=256, w_scale=sc)
    assert h.w_scale == pytest.approx(sc, rel=1e-6)
    p4, s4, z4 = inputs.quant_awq4_weights(inputs.weights_f32(128, 512, seed=13, outliers=False), 128)
    _, st, _, side = _roundtrip(oc.FMT_INT4_AWQ, p4, 512, tile_k=256, scales=s4, zeros=z4, group_size=128)
    assert np.array_equal(side["scales"], s4) and np.array_equal(side["zeros"], z4)
    assert st["bits_per_weight"] >= st["h_sym_bits_per_weight"]


def test_roundtrip_degenerate_constant_matrix():
    w = np.full((128, 64), 0x3C00, dtype=np.uint16)
    _roundtrip(oc.FMT_BF16, w, 64)
    _roundtrip(oc.FMT_BF16, w, 64, flags=oc.FLAG_STATE_PAYLOAD)
    _roundtrip(oc.FMT_INT8, np.zeros((128, 256), dtype=np.int8), 256, scales=np.ones(128, np.float16))


def test_tiles_are_independently_decodable():
    """Random access (P:l.127, l.149, l.167): decoding one tile needs only its record + the table."""
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(256, 256, seed=14))
    buf, _ = oc.encode(oc.FMT_BF16, w, 256, tile_k=64)
    h = oc.Header.unpack(buf)
    f = np.frombuffer(buf[h.off_freq:h.off_freq + 512].tobytes(), dtype="<u2").astype(np.uint32)
    tab = codec.Table(f, 12)
    off = np.frombuffer(buf[h.off_offsets:h.off_offsets + 4 * (h.n_tiles + 1)].tobytes(), dtype="<u4").astype(np.int64)
    rows, cols = oc.tile_order(oc.FMT_BF16, 64)
    coded, _ = oc.symbolise(oc.FMT_BF16, w)
    for t in (5, 0, 7, 2):
        a, e = h.off_records + 16 * off[t], h.off_records + 16 * off[t + 1]
        states = np.frombuffer(buf[a:a + 128].tobytes(), dtype="<u4").astype(np.uint64)
        words = np.frombuffer(buf[a + 128:e].tobytes(), dtype="<u2")
        sym, end, _ = codec.tile_decode(states, words, 8192, 32, tab, 16, 16)
        stripe, kt = divmod(t, 4)
        assert np.array_equal(sym, coded[stripe * 128:(stripe + 1) * 128, kt * 64:(kt + 1) * 64][rows, cols])
        assert np.all(end == 65536)


def test_corrupt_container_is_detected():
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(128, 128, seed=15))
    buf, _ = oc.encode(oc.FMT_BF16, w, 128, tile_k=64)
    h = oc.Header.unpack(buf)
    bad = buf.copy()
    bad[h.off_records + 3] ^= 0x40            # flip a bit of lane 0's start state
    with pytest.raises(ValueError):
        _, w2, _ = oc.decode(bad)


# ------------------------------------------------------------------------------------------------
def test_e4m3_decode_against_torch_cast():
    import torch
    codes = np.arange(256, dtype=np.uint8)
    ref = torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    got = og.e4m3_to_f64(codes)
    assert np.array_equal(np.isnan(ref), np.isnan(got))
    ok = ~np.isnan(ref)
    assert np.array_equal(ref[ok], got[ok])
    assert got[0x7E] == 448.0 and got[0x01] == 2.0 ** -9


def test_e5m2_decode_against_binary16_and_torch():
    """e5m2 is the upper byte of an IEEE binary16 (pin 1: numpy's float16) and torch's float8_e5m2 (pin 2)."""
    import torch
    codes = np.arange(256, dtype=np.uint8)
    got = og.e5m2_to_f64(codes)
    ref16 = (codes.astype(np.uint16) << 8).view(np.float16).astype(np.float64)
    ref_t = torch.from_numpy(codes).view(torch.float8_e5m2).to(torch.float64).numpy()
    for ref in (ref16, ref_t):
        assert np.array_equal(np.isnan(ref), np.isnan(got))
        ok = ~np.isnan(ref)
        assert np.array_equal(ref[ok], got[ok])
    assert got[0x7B] == 57344.0 and got[0x01] == 2.0 ** -16 and got[0x3C] == 1.0 and got[0xFC] == -np.inf


def test_roundtrip_and_gemm_fp8_e5m2():
    f8, sc = inputs.quant_fp8_e5m2_weights(inputs.weights_f32(128, 512, seed=14, std=0.015, outliers=False))
    _, st, h, _ = _roundtrip(oc.FMT_FP8_E5M2, f8, 512, tile_k=256, w_scale=sc)
    assert h.fmt == oc.FMT_FP8_E5M2 and st["bits_per_weight"] < 8.0
    x8 = np.array([[0x3C, 0x40, 0xBC, 0x00]], np.uint8)       # 1, 2, -1, 0 in e5m2
    w8 = np.array([[0x38, 0x38, 0x38, 0x7B]], np.uint8)       # 0.5, 0.5, 0.5, 57344
    y, a = og.gemm_fp8(x8, np.array([2.0], np.float32), w8, 0.5, x_e5m2=True, w_e5m2=True)
    assert y[0, 0] == (0.5 + 1.0 - 0.5) * 2.0 * 0.5 and a[0, 0] == 2.0 * 2.0 * 0.5
    # mixed kinds: the same bytes read as e4m3 give 1.5 / 2 / -1.5 (0x3C = 1.5 in e4m3, 0x40 = 2)
    y, _ = og.gemm_fp8(x8, np.array([1.0], np.float32), w8, 1.0, x_e5m2=False, w_e5m2=True)
    assert y[0, 0] == (1.5 + 2.0 - 1.5) * 0.5


def test_e2m1_values_and_fp4_roundtrip():
    """fp4-e2m1 (P:l.80): the 16 code values of the OCP table; each is exactly an e4m3 number (what the kernel
    feeds the tensor core), checked through torch's e4m3 cast; container round trip; quantiser sanity."""
    import torch
    got = og.e2m1_to_f64(np.arange(16))
    table = [0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0]
    assert got.tolist() == table + [-v for v in table] and np.signbit(got[8])
    back = torch.from_numpy(got.astype(np.float32)).to(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert np.array_equal(back, got)
    wf = inputs.weights_f32(128, 512, seed=15, outliers=False)
    p4, sc = inputs.quant_fp4_weights(wf)
    _, st, h, _ = _roundtrip(oc.FMT_FP4_E2M1, p4, 512, tile_k=256, w_scale=sc)
    assert h.w_scale == pytest.approx(sc, rel=1e-6) and st["payload_bits"] / st["n_weights"] < 4.0
    wd = og.e2m1_to_f64(og.int4_unpack(p4)) * sc
    assert np.all(np.abs(wd - wf) <= 1.0 * sc + 1e-9)           # largest grid gap is 2 (4 -> 6): half of it
    x8 = np.array([[0x38, 0x40]], np.uint8)                      # 1.0, 2.0 in e4m3
    y, a = og.gemm_fp4(x8, np.array([2.0], np.float32), np.array([[0x7A]], np.uint8), 0.5)   # codes 0xA = -1.0, 0x7 = 6.0
    assert y[0, 0] == (1.0 * -1.0 + 2.0 * 6.0) * 2.0 * 0.5 and a[0, 0] == 13.0


def test_pair_variant_stream_and_container():
    """S: 8(f) NEXT-5 bf16 pair variant.  Pins: without escapes the literal-carrying stream IS the plain rANS stream;
    with escapes it round-trips and every literal comes back at its nibble; the container is lossless, carries its
    code table, and costs within 0.03 bit/weight of the one-symbol-per-weight bf16 container."""
    rng = np.random.default_rng(5)
    codes = rng.choice(16, size=512, p=np.r_[np.full(15, 0.98 / 15), 0.02])
    sym = (codes[0::2] | (codes[1::2] << 4)).astype(np.uint8)
    tab = codec.Table(codec.normalize(codec.histogram(sym), 12), 12)
    lits = rng.integers(0, 256, size=int((codes == 15).sum()))
    st, words, after = codec.encode_scalar_lit(sym, tab, 16, 16, 65536 + 77, lits)
    o, l, end, used = codec.decode_scalar_lit(st, words, sym.size, tab, 16, 16)
    assert np.array_equal(o, sym) and end == 65536 + 77 and used == words.size == after[-1]
    assert np.array_equal(l[l != 0xFFFF], lits) and np.array_equal(np.flatnonzero(l != 0xFFFF), np.flatnonzero(codes == 15))
    assert np.all(np.diff(after.astype(np.int64)) >= 0)
    calm = (np.minimum(sym & 15, 14) | (np.minimum(sym >> 4, 14) << 4)).astype(np.uint8)
    tab2 = codec.Table(codec.normalize(codec.histogram(calm), 12), 12)
    s1, w1 = codec.encode_scalar(calm, tab2, 16, 16, 65536)
    s2, w2, _ = codec.encode_scalar_lit(calm, tab2, 16, 16, 65536, [])
    assert s1 == s2 and np.array_equal(w1, w2)
    w = inputs.f32_to_bf16_bits(inputs.weights_f32(256, 512, seed=16, jitter=True)).copy()
    w[5, 17], w[200, 300], w[200, 301] = 0x0001, 0x7F7F, 0x0080
    coded, raw, exps, table = oc.symbolise_pair(w)
    cnt = np.bincount(exps.ravel(), minlength=256)
    assert len(set(table[:15].tolist())) == 15 and min(cnt[table[:15]]) >= max(np.delete(cnt, table[:15]))
    buf, st = _roundtrip(oc.FMT_BF16_PAIR4, w, 512, tile_k=256, flags=3, tile_n=32)[:2]
    _, st0 = oc.encode(oc.FMT_BF16, w, 512, tile_k=256, flags=3, tile_n=32)
    assert 0.0 <= st["bits_per_weight"] - st0["bits_per_weight"] <= 0.03
    h = oc.Header.unpack(buf)
    assert np.array_equal(buf[h.off_zeros:h.off_zeros + 16], table)


def test_bf16_conversion_against_torch():
    import torch
    x = np.random.default_rng(1).standard_normal(4096).astype(np.float32) * 3
    bits = inputs.f32_to_bf16_bits(x)
    ref = torch.from_numpy(x).to(torch.bfloat16)
    assert np.array_equal(bits, ref.view(torch.int16).numpy().view(np.uint16))
    assert np.array_equal(og.bf16_bits_to_f64(bits), ref.to(torch.float64).numpy())


def test_gemm_brute_force_and_unit_vector():
    rng = np.random.default_rng(2)
    wb = inputs.f32_to_bf16_bits(rng.standard_normal((6, 10)).astype(np.float32))
    xb = inputs.f32_to_bf16_bits(rng.standard_normal((3, 10)).astype(np.float32))
    y, a = og.gemm_bf16(xb, wb)
    wf, xf = og.bf16_bits_to_f64(wb), og.bf16_bits_to_f64(xb)
    for m in range(3):
        for n in range(6):
            acc = sum(float(xf[m, k]) * float(wf[n, k]) for k in range(10))
            assert y[m, n] == pytest.approx(acc, rel=1e-12, abs=1e-15)
            assert a[m, n] == pytest.approx(sum(abs(float(xf[m, k]) * float(wf[n, k])) for k in range(10)), rel=1e-12)
    e = np.zeros((1, 10), dtype=np.float32); e[0, 7] = 1.0
    y, _ = og.gemm_bf16(inputs.f32_to_bf16_bits(e), wb)
    assert np.array_equal(y[0], wf[:, 7])        # Y = column 7 of W exactly


def test_gemm_int8_int4_fp8_definitions():
    rng = np.random.default_rng(3)
    wq = rng.integers(-127, 128, size=(5, 64)).astype(np.int8)
    xq = rng.integers(-127, 128, size=(2, 64)).astype(np.int8)
    sw = rng.uniform(0.001, 0.01, 5).astype(np.float16)
    sx = rng.uniform(0.01, 0.1, 2).astype(np.float32)
    y, a, acc = og.gemm_int8(xq, sx, wq, sw)
    for m in range(2):
        for n in range(5):
            s = sum(int(xq[m, k]) * int(wq[n, k]) for k in range(64))
            assert acc[m, n] == s
            assert y[m, n] == s * float(sx[m]) * float(sw[n])
    packed = rng.integers(0, 256, size=(4, 64)).astype(np.uint8)       # k = 128
    sc = rng.uniform(0.001, 0.01, (4, 1)).astype(np.float16)
    zr = rng.integers(0, 16, (4, 1)).astype(np.float16)
    wd = og.awq_dequant_f64(packed, sc, zr, 128)
    assert wd[2, 10] == ((int(packed[2, 5]) & 15) - float(zr[2, 0])) * float(sc[2, 0])
    assert wd[2, 11] == ((int(packed[2, 5]) >> 4) - float(zr[2, 0])) * float(sc[2, 0])
    x8 = rng.integers(0, 0x7F, size=(2, 32)).astype(np.uint8)
    w8 = rng.integers(0, 0x7F, size=(3, 32)).astype(np.uint8)
    y, _ = og.gemm_fp8(x8, np.array([2.0, 0.5], np.float32), w8, 0.25)
    ref = (og.e4m3_to_f64(x8) @ og.e4m3_to_f64(w8).T) * np.array([[0.5], [0.125]])
    assert np.allclose(y, ref, rtol=1e-14)


def test_quantisers_reconstruct_within_half_step():
    """Input recipe sanity (A13/A14): the quantisers behave like round-to-nearest on their grids."""
    wf = inputs.weights_f32(128, 256, seed=21, jitter=True)
    q, s = inputs.quant_sq8_weights(wf)
    err = np.abs(q.astype(np.float32) * s.astype(np.float32)[:, None] - wf)
    assert np.all(err <= 0.51 * s.astype(np.float32)[:, None] + 1e-7)
    p, sc, z = inputs.quant_awq4_weights(wf, 128)
    wd = og.awq_dequant_f64(p, sc, z, 128)
    assert np.all(np.abs(wd - wf) <= 1.01 * np.repeat(sc.astype(np.float64), 128, axis=1))
    rows, tok = inputs.route_top2(20, 8, seed=5)
    assert rows.sum() == 40 and np.all(np.bincount(tok, minlength=20) == 2)
