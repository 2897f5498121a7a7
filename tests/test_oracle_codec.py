"""Pins for the oracle's codec (oracle/anslin_oracle.c) against what the paper and the mathematics
fix — none of them re-types the oracle's own formula.  CPU only."""
import itertools
import math
import os

import numpy as np
import pytest

from oracle import codec

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _load_example(name):
    d = {"table": []}
    for line in open(os.path.join(GOLD, name)):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, *v = line.split()
        v = [int(t) for t in v]
        if k == "table":
            d["table"].append(v)
        else:
            d[k] = v if len(v) > 1 or k in ("message", "words", "enc_states", "dec_states") else v[0]
    f = np.zeros(256, dtype=np.uint32)
    for s, fs, cs in d["table"]:
        f[s] = fs
    d["tab"] = codec.Table(f, d["b"])
    for s, fs, cs in d["table"]:
        assert d["tab"].c[s] == cs          # the example's cumulative column
    return d


@pytest.mark.parametrize("name", ["example_a.txt", "example_b.txt"])
def test_worked_examples(name):
    """Hand-worked values (tests/golden/example_*.txt; P:l.268-285 Alg V.2, ref [13])."""
    d = _load_example(name)
    msg, tab = np.array(d["message"], dtype=np.uint8), d["tab"]
    state, words = codec.encode_scalar(msg, tab, d["w"], d["Llog2"], d["x_init"])
    assert state == d["state"]
    assert list(words) == d["words"]
    # every intermediate encoder state: encoding the last j symbols alone ends in enc_states[j-1]
    for j in range(1, len(msg) + 1):
        st, _ = codec.encode_scalar(msg[len(msg) - j:], tab, d["w"], d["Llog2"], d["x_init"])
        assert st == d["enc_states"][j - 1]
    out, end, used = codec.decode_scalar(d["state"], d["words"], len(msg), tab, d["w"], d["Llog2"])
    assert list(out) == d["message"] and end == d["x_init"] and used == len(d["words"])
    for j in range(1, len(msg) + 1):
        _, st, _ = codec.decode_scalar(d["state"], d["words"], j, tab, d["w"], d["Llog2"])
        assert st == d["dec_states"][j - 1]


def test_power_of_two_closed_form():
    """All f powers of two => rANS degenerates to a prefix code: every step grows the bit length of
    the state by exactly log2(M/f), so bitlen(x_final) + w*#words = bitlen(L) + sum log2(M/f_i)."""
    rng = np.random.default_rng(3)
    b, w, Ll = 12, 16, 16
    f = np.zeros(256, dtype=np.uint32)
    f[[0, 1, 2, 3, 4, 5]] = [2048, 1024, 512, 256, 128, 128]
    tab = codec.Table(f, b)
    for n in (1, 7, 100, 1000):
        msg = rng.choice(6, size=n, p=f[:6] / 4096.0).astype(np.uint8)
        state, words = codec.encode_scalar(msg, tab, w, Ll, 1 << Ll)
        bits = sum(b - int(math.log2(f[s])) for s in msg)
        assert state.bit_length() + w * len(words) == (Ll + 1) + bits


def test_uniform_table_special_case():
    """256 symbols, f = 16 each: every symbol costs exactly 8 bits, i.e. one 16-bit word per two
    symbols (+-1 at the ends) and the decoded bytes are literally the state's digits."""
    rng = np.random.default_rng(4)
    tab = codec.Table(np.full(256, 16, dtype=np.uint32), 12)
    for n in (2, 64, 1001):
        msg = rng.integers(0, 256, size=n).astype(np.uint8)
        state, words = codec.encode_scalar(msg, tab, 16, 16, 1 << 16)
        assert abs(len(words) - n / 2) <= 1
        assert state.bit_length() + 16 * len(words) == 17 + 8 * n
        out, end, used = codec.decode_scalar(state, words, n, tab, 16, 16)
        assert np.array_equal(out, msg) and end == 1 << 16 and used == len(words)


def test_brute_force_tiny_alphabet():
    """M = 16, every message of length <= 6 over 3 symbols: round trip and unique decodability
    (distinct messages of one length never share (state, words))."""
    f = np.zeros(256, dtype=np.uint32)
    f[:3] = [8, 5, 3]
    tab = codec.Table(f, 4)
    for n in range(1, 7):
        seen = {}
        for msg in itertools.product(range(3), repeat=n):
            m = np.array(msg, dtype=np.uint8)
            state, words = codec.encode_scalar(m, tab, 4, 4, 16)
            assert 16 <= state < 256 and all(0 <= x < 16 for x in words)
            key = (state, tuple(words))
            assert key not in seen, (msg, seen.get(key))
            seen[key] = msg
            out, end, used = codec.decode_scalar(state, words, n, tab, 4, 4)
            assert tuple(out) == msg and end == 16 and used == len(words)


@pytest.mark.parametrize("x_init", [1 << 16, (1 << 16) + 0xBEEF, (1 << 17) - 1])
def test_final_state_invariant_and_arbitrary_init(x_init):
    """'ANS supports arbitrary initial states' (P:l.167): after the last symbol the decoder state is
    the encoder's start state, whatever it was in [L, 2L)."""
    rng = np.random.default_rng(5)
    cnt = np.bincount(rng.geometric(0.3, size=5000).clip(0, 255), minlength=256).astype(np.uint64)
    tab = codec.Table(codec.normalize(cnt, 12), 12)
    live = np.flatnonzero(cnt)
    msg = rng.choice(live, size=777).astype(np.uint8)
    state, words = codec.encode_scalar(msg, tab, 16, 16, x_init)
    assert (1 << 16) <= state < (1 << 32)
    out, end, used = codec.decode_scalar(state, words, msg.size, tab, 16, 16)
    assert np.array_equal(out, msg) and end == x_init and used == len(words)


def test_interleave_two_formulations_and_lane_independence():
    """32-lane tile: (i) the backward shared-stack encoder and the decoder-simulation encoder give
    the same bytes; (ii) tile decode == 32 independent scalar decodes of the lane streams (P:l.192)."""
    rng = np.random.default_rng(6)
    cnt = np.bincount(rng.geometric(0.25, size=20000).clip(0, 255), minlength=256).astype(np.uint64)
    tab = codec.Table(codec.normalize(cnt, 12), 12)
    live = np.flatnonzero(cnt)
    R, steps = 32, 40
    sym = rng.choice(live, size=R * steps, p=cnt[live] / cnt.sum()).astype(np.uint8)
    x_init = (1 << 16) + rng.integers(0, 1 << 16, size=R).astype(np.uint64)
    st1, w1 = codec.tile_encode(sym, R, tab, 16, 16, x_init)
    st2, w2 = codec.tile_encode(sym, R, tab, 16, 16, x_init, by_simulation=True)
    assert np.array_equal(st1, st2) and np.array_equal(w1, w2)
    out, end, used = codec.tile_decode(st1, w1, sym.size, R, tab, 16, 16)
    assert np.array_equal(out, sym) and np.array_equal(end, x_init) and used == len(w1)
    total = 0
    for lane in range(R):
        ls = sym[lane::R]
        s, w = codec.encode_scalar(ls, tab, 16, 16, int(x_init[lane]))
        assert s == int(st1[lane])
        o, e, u = codec.decode_scalar(s, w, ls.size, tab, 16, 16)
        assert np.array_equal(o, ls) and e == int(x_init[lane])
        total += len(w)
    assert total == len(w1)


def test_normalise_invariants():
    rng = np.random.default_rng(7)
    for trial in range(20):
        k = int(rng.integers(2, 257))
        cnt = np.zeros(256, dtype=np.uint64)
        idx = rng.choice(256, size=k, replace=False)
        cnt[idx] = (rng.pareto(1.0, size=k) * 50 + 1).astype(np.uint64)
        f = codec.normalize(cnt, 12)
        assert int(f.sum()) == 4096
        assert np.array_equal(f > 0, cnt > 0)
        H, X = codec.entropy(cnt), codec.cross_entropy(cnt, f, 12)
        assert X >= H - 1e-12                      # Gibbs' inequality
        assert X - H < 0.08                        # 12-bit quantisation loss stays small
    # a table that already sums to 4096 is its own optimum
    f0 = np.zeros(256, dtype=np.uint64); f0[:4] = [2048, 1024, 512, 512]
    assert np.array_equal(codec.normalize(f0, 12), f0.astype(np.uint32))


def test_normalise_degenerate_single_symbol():
    """Reading A11: one live symbol -> f = 4095 for it, 1 for its successor; still round-trips."""
    cnt = np.zeros(256, dtype=np.uint64); cnt[255] = 1000
    f = codec.normalize(cnt, 12)
    assert f[255] == 4095 and f[0] == 1 and int(f.sum()) == 4096
    tab = codec.Table(f, 12)
    msg = np.full(500, 255, dtype=np.uint8)
    s, w = codec.encode_scalar(msg, tab, 16, 16, 1 << 16)
    out, end, _ = codec.decode_scalar(s, w, 500, tab, 16, 16)
    assert np.array_equal(out, msg) and end == 1 << 16 and len(w) <= 1


def test_entropy_against_library_and_closed_forms():
    from scipy.stats import entropy as sp_entropy
    rng = np.random.default_rng(8)
    cnt = rng.integers(0, 1000, size=256).astype(np.uint64)
    assert codec.entropy(cnt) == pytest.approx(sp_entropy(cnt.astype(float), base=2), abs=1e-12)
    assert codec.entropy(np.full(256, 7, dtype=np.uint64)) == pytest.approx(8.0, abs=1e-12)
    two = np.zeros(256, dtype=np.uint64); two[3], two[200] = 1, 3
    assert codec.entropy(two) == pytest.approx(-(0.25 * math.log2(0.25) + 0.75 * math.log2(0.75)), abs=1e-12)
    sym = rng.integers(0, 256, size=10000).astype(np.uint8)
    assert np.array_equal(codec.histogram(sym), np.bincount(sym, minlength=256).astype(np.uint64))


def test_compressed_size_tracks_entropy():
    """Achieved bits >= n*H of the message's own histogram can fail only by the table mismatch;
    against the TABLE's cross entropy the rANS payload is within the flush cost (P:l.349)."""
    rng = np.random.default_rng(9)
    cnt = np.bincount(rng.geometric(0.2, size=100000).clip(0, 255), minlength=256).astype(np.uint64)
    f = codec.normalize(cnt, 12)
    tab = codec.Table(f, 12)
    live = np.flatnonzero(cnt)
    msg = rng.choice(live, size=50000, p=cnt[live] / cnt.sum()).astype(np.uint8)
    state, words = codec.encode_scalar(msg, tab, 16, 16, 1 << 16)
    ideal = float(np.sum(np.log2(4096.0 / f[msg])))
    written = 32 + 16 * len(words)
    assert ideal <= written <= ideal + 32 + 0.001 * ideal


# ------------------------------------------------------------------------------------------------
# Property tests (hypothesis): any histogram, any stream, any legal start state
# ------------------------------------------------------------------------------------------------
from hypothesis import given, settings, strategies as st_


@settings(max_examples=60, deadline=None)
@given(st_.lists(st_.integers(0, 255), min_size=1, max_size=600), st_.integers(0, 0xFFFF))
def test_property_scalar_round_trip_and_size(sym_list, payload):
    """For ANY symbol sequence: the scalar rANS stream decodes to the sequence, ends in its start state (any state in
    [L, 2L) is a legal start, reading A4), and its size is within the coder's worst case of the table's cross entropy."""
    sym = np.array(sym_list, dtype=np.uint8)
    cnt = codec.histogram(sym)
    f = codec.normalize(cnt, 12)
    assert int(f.sum()) == 4096 and np.all(f[cnt > 0] >= 1) and np.all(f[cnt == 0] == 0) | (np.count_nonzero(cnt) == 1)
    tab = codec.Table(f, 12)
    x_init = (1 << 16) + payload
    state, words = codec.encode_scalar(sym, tab, 16, 16, x_init)
    out, end, used = codec.decode_scalar(state, words, sym.size, tab, 16, 16)
    assert np.array_equal(out, sym) and end == x_init and used == words.size
    assert (1 << 16) <= state < (1 << 32)
    ideal = codec.cross_entropy(cnt, f, 12) * sym.size          # bits
    assert 16 * words.size + 32 >= ideal - 1e-6                 # never below the table's own bound (state bits included)
    assert 16 * words.size <= ideal + 32 + 16                   # at most the start state's bits and one word of slack above it


@settings(max_examples=40, deadline=None)
@given(st_.lists(st_.integers(0, 15), min_size=8, max_size=512).filter(lambda v: len(v) % 8 == 0), st_.data())
def test_property_pair_stream_with_literals(code_list, data):
    """bf16 pair variant's lane stream: for ANY sequence of 4-bit codes (15 = escape) and ANY literals the stream round
    trips, every literal returns at its own nibble, and literal words sit after the renormalisation of their 4-step chunk."""
    codes = np.array(code_list, dtype=np.uint8)
    sym = (codes[0::2] | (codes[1::2] << 4)).astype(np.uint8)
    n_esc = int((codes == 15).sum())
    lits = np.array(data.draw(st_.lists(st_.integers(0, 255), min_size=n_esc, max_size=n_esc)), dtype=np.uint16)
    tab = codec.Table(codec.normalize(codec.histogram(sym), 12), 12)
    state, words, after = codec.encode_scalar_lit(sym, tab, 16, 16, 1 << 16, lits)
    out, lit, end, used = codec.decode_scalar_lit(state, words, sym.size, tab, 16, 16)
    assert np.array_equal(out, sym) and end == (1 << 16) and used == words.size == int(after[-1])
    assert np.array_equal(lit[codes == 15], lits) and np.all(lit[codes != 15] == 0xFFFF)
    plain_state, plain_words = codec.encode_scalar(sym, tab, 16, 16, 1 << 16)
    assert plain_state == state and words.size == plain_words.size + n_esc       # literals are the only extra words
    # the words consumed inside a chunk before its last step never include that chunk's literals
    esc_per_chunk = (codes.reshape(-1, 8) == 15).sum(axis=1)
    rn = np.diff(np.concatenate([[0], after.astype(np.int64)]))
    assert np.all(rn.reshape(-1, 4)[:, :3] <= 1) and np.all(rn.reshape(-1, 4)[:, 3] <= 1 + esc_per_chunk)
