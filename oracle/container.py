"""ORACLE (test infrastructure only) — symbolisation, tile order and the compressed container.

Follows the paper's offline stage (P:l.165-169 §V-B, P:l.149 §IV): whole-matrix histogram ->
one shared codebook -> partition into GEMM tiles -> each tile entropy-coded as R=32 interleaved
rANS streams with independently initialised states -> bitstream + 4-byte tile offsets.
The byte layout is the one DESIGN.md §"Container" states (the paper gives only Eq.3, P:l.440);
nothing here is shared with the product encoder in paper_2606_15789_b200/csrc.

Parity note: container BYTES are "parity unpinned" by the paper (any legal table / tie-break is
correct).  What is pinned: decode(encode(W)) == W bit for bit (P:l.26, l.46, l.486), the size
bound against the entropy (P:l.12, l.349) and Eq.3's metadata (P:l.440-466).
"""
from __future__ import annotations

import struct
from dataclasses import dataclass

import numpy as np

from . import codec

MAGIC = 0x4C534E41  # "ANSL"
VERSION = 1
FMT_BF16, FMT_FP8_E4M3, FMT_INT8, FMT_INT4_AWQ, FMT_FP8_E5M2, FMT_FP4_E2M1, FMT_BF16_PAIR4 = 0, 1, 2, 3, 4, 5, 6
FLAG_STATE_PAYLOAD = 1
FLAG_LANE_STREAMS = 2   # each lane's words stored as its own stream (tile_n = 32 only), see _lane_record
SEG_STEPS = 256         # lane-stream records are cut into segments of this many decode steps
STRIPE_N = 128        # weight rows per stripe = MMA M; a stripe is cut into tiles of tile_n rows
TILE_N = 128          # default tile_n (BASELINE config 1: 128 x 64 tiles); 32 is the other supported height
LANES = 32            # R interleaved streams per tile (P:l.192; BASELINE config 1)
PROB_BITS = 12        # b (P:l.442 "default b = 12")
WORD_BITS = 16        # w   (reading A3)
STATE_LO_LOG2 = 16    # L = 2^16 (reading A3)
HEADER_BYTES = 128
TAIL_BYTES = 4096      # readable bytes that must follow the records section

# symbols per 16-byte operand chunk, and default tile_k (in weights) per format
SPC = {FMT_BF16: 8, FMT_FP8_E4M3: 16, FMT_INT8: 16, FMT_INT4_AWQ: 4, FMT_FP8_E5M2: 16, FMT_FP4_E2M1: 8, FMT_BF16_PAIR4: 4}
DEFAULT_TILE_K = {FMT_BF16: 64, FMT_FP8_E4M3: 256, FMT_INT8: 256, FMT_INT4_AWQ: 256, FMT_FP8_E5M2: 256, FMT_FP4_E2M1: 256, FMT_BF16_PAIR4: 256}
WEIGHTS_PER_SYMBOL = {FMT_BF16: 1, FMT_FP8_E4M3: 1, FMT_INT8: 1, FMT_INT4_AWQ: 2, FMT_FP8_E5M2: 1, FMT_FP4_E2M1: 2, FMT_BF16_PAIR4: 2}


def seg_steps(fmt: int) -> int:
    """Decode steps per lane-stream segment: 256 where a symbol carries few bits (bf16 exponents, SQ8), 128 where it
    carries 6-7 bits (fp8, packed 4-bit pairs, bf16 exponent pairs): a segment is what the decoder stages at once."""
    return SEG_STEPS if fmt in (FMT_BF16, FMT_INT8) else SEG_STEPS // 2


def _align(x: int, a: int = 16) -> int:
    return (x + a - 1) // a * a


# ---------------------------------------------------------------------------------------------
# Symbolisation (reading A1): which 8-bit symbol stands for which bits of a weight.
# ---------------------------------------------------------------------------------------------
def symbolise(fmt: int, w: np.ndarray):
    """Returns (coded symbol matrix uint8 [n_out x sym_cols], raw plane matrix or None).

    bf16 (w: uint16 bit patterns [n_out x k_in]): coded symbol = exponent bits 14..7;
        raw byte = (mantissa bits 6..0) << 1 | sign bit 15  (bf16 rotated left by one, low byte).
    fp8 / int8 (w: uint8 / int8 [n_out x k_in]): the byte itself.
    int4 / fp4 (w: uint8 [n_out x k_in/2], low nibble = even k): the packed byte (two K-adjacent codes).
    """
    if fmt == FMT_BF16:
        w = np.ascontiguousarray(w).view(np.uint16)
        coded = ((w >> 7) & 0xFF).astype(np.uint8)
        raw = (((w & 0x7F) << 1) | (w >> 15)).astype(np.uint8)
        return coded, raw
    return np.ascontiguousarray(w).view(np.uint8), None


def pair_code_table(exps: np.ndarray) -> np.ndarray:
    """bf16 pair variant (S: 8(f) NEXT-5): the 15 most frequent exponent bytes get the 4-bit codes 0..14 (descending
    count, ties by smaller exponent); code 15 is the escape.  Returns uint8[16], entry 15 = 0."""
    cnt = np.bincount(exps.ravel(), minlength=256)
    order = sorted(range(256), key=lambda v: (-int(cnt[v]), v))[:15]
    return np.array(order + [0], dtype=np.uint8)


def symbolise_pair(w: np.ndarray, table: np.ndarray | None = None):
    """bf16 -> (coded pairs uint8 [n x k/2] = code(even k) | code(odd k) << 4, raw plane uint8 [n x k] as for bf16,
    exponent bytes uint8 [n x k], code table uint8[16])."""
    w = np.ascontiguousarray(w).view(np.uint16)
    exps = ((w >> 7) & 0xFF).astype(np.uint8)
    raw = (((w & 0x7F) << 1) | (w >> 15)).astype(np.uint8)
    table = pair_code_table(exps) if table is None else table
    code_of = np.full(256, 15, dtype=np.uint8)
    code_of[table[:15]] = np.arange(15, dtype=np.uint8)
    codes = code_of[exps]
    return (codes[:, 0::2] | (codes[:, 1::2] << 4)).astype(np.uint8), raw, exps, table


def desymbolise(fmt: int, coded: np.ndarray, raw):
    if fmt == FMT_BF16:
        c = coded.astype(np.uint16)
        r = raw.astype(np.uint16)
        return ((r & 1) << 15) | (c << 7) | (r >> 1)
    return coded


def tile_order(fmt: int, tile_k: int, tile_n: int = TILE_N):
    """Tile symbol order (reading A6).  Returns (rows, cols): symbol i of the tile is the coded
    symbol at (row rows[i], symbol column cols[i]) of the tile's [tile_n x sym_cols] symbol matrix.

    i = t*32 + lane.  The tile is cut along K into units of 32 operand bytes per row
    (16 bf16/fp16 weights, 32 fp8/int8 weights; fp4 is expanded to one e4m3 byte per weight: 32 weights);
    unit u is decoded completely before unit u+1.
    Inside a unit there are G = 2*tile_n/32 chunk rounds g; in round g lane l owns the 16-byte
    operand chunk (row (g mod tile_n/32)*32 + l, half g div (tile_n/32)) and produces its spc
    symbols in steps t = (u*G + g)*spc + e, e = 0..spc-1.  (tile_n = 32: lane l simply walks row l.)
    """
    assert tile_n in (32, 128)
    spc = SPC[fmt]
    rb = tile_n // 32
    G = 2 * rb
    sym_cols = tile_k // WEIGHTS_PER_SYMBOL[fmt]
    units = sym_cols // (2 * spc)
    assert units * 2 * spc == sym_cols, "tile_k must be a multiple of the unit width"
    steps = units * G * spc
    rows = np.zeros(steps * LANES, dtype=np.int64)
    cols = np.zeros(steps * LANES, dtype=np.int64)
    for u in range(units):
        for g in range(G):
            for e in range(spc):
                t = (u * G + g) * spc + e
                for lane in range(LANES):
                    rows[t * LANES + lane] = (g % rb) * 32 + lane
                    cols[t * LANES + lane] = u * 2 * spc + (g // rb) * spc + e
    return rows, cols


# ---------------------------------------------------------------------------------------------
@dataclass
class Header:
    fmt: int
    n_out: int
    k_in: int
    tile_n: int
    tile_k: int
    streams: int
    prob_bits: int
    word_bits: int
    state_lo_log2: int
    group_size: int
    flags: int
    n_tiles: int
    w_scale: float
    off_freq: int
    off_offsets: int
    off_records: int
    off_raw: int
    off_scales: int
    off_zeros: int
    total_bytes: int

    max_seg_bytes: int = 0      # lane-stream layout: shared-memory bytes the largest segment needs when staged

    def pack(self) -> bytes:
        return struct.pack("<14IfI8Q", MAGIC, VERSION, self.fmt, self.n_out, self.k_in, self.tile_n, self.tile_k,
                           self.streams, self.prob_bits, self.word_bits, self.state_lo_log2, self.group_size,
                           self.flags, self.n_tiles, self.w_scale, self.max_seg_bytes, self.off_freq, self.off_offsets,
                           self.off_records, self.off_raw, self.off_scales, self.off_zeros, self.total_bytes, 0)

    @staticmethod
    def unpack(buf) -> "Header":
        v = struct.unpack("<14IfI8Q", bytes(buf[:HEADER_BYTES]))
        if v[0] != MAGIC or v[1] != VERSION:
            raise ValueError("not an anslin container")
        return Header(*v[2:15], *v[16:23], max_seg_bytes=v[15])


def raw_tile_bytes(tile_k: int, flags: int, tile_n: int = TILE_N) -> int:
    n = tile_n * tile_k
    return n - 64 if flags & FLAG_STATE_PAYLOAD else n


def _raw_tile_pack(raw_lane_major: np.ndarray, flags: int):
    """raw_lane_major: uint8 [steps x 32] raw bytes in tile order.  Returns (plane bytes, payload[32]).

    Plane layout: 16-step vectors; vector v of lane l at v*512 + l*16.  With the state-payload flag
    the two raw bytes of each lane's last two steps ride in the rANS start state (reading A4) and
    the last vector is stored as 7 sub-rows of 32 x 2 bytes.
    """
    steps = raw_lane_major.shape[0]
    V = steps // 16
    vec = raw_lane_major.reshape(V, 16, LANES).transpose(0, 2, 1)          # [v][lane][pos]
    if not flags & FLAG_STATE_PAYLOAD:
        return vec.reshape(-1).copy(), np.zeros(LANES, dtype=np.uint64)
    head = vec[:V - 1].reshape(-1)
    last = vec[V - 1]                                                      # [lane][16]
    sub = last[:, :14].reshape(LANES, 7, 2).transpose(1, 0, 2).reshape(-1)  # [h][lane][2]
    payload = last[:, 14].astype(np.uint64) | (last[:, 15].astype(np.uint64) << 8)
    return np.concatenate([head, sub]), payload


def _raw_tile_unpack(plane: np.ndarray, steps: int, flags: int, payload):
    V = steps // 16
    if not flags & FLAG_STATE_PAYLOAD:
        return plane.reshape(V, LANES, 16).transpose(0, 2, 1).reshape(steps, LANES)
    vec = np.zeros((V, LANES, 16), dtype=np.uint8)
    vec[:V - 1] = plane[:(V - 1) * 512].reshape(V - 1, LANES, 16)
    sub = plane[(V - 1) * 512:].reshape(7, LANES, 2).transpose(1, 0, 2).reshape(LANES, 14)
    vec[V - 1, :, :14] = sub
    vec[V - 1, :, 14] = (payload & 0xFF).astype(np.uint8)
    vec[V - 1, :, 15] = ((payload >> 8) & 0xFF).astype(np.uint8)
    return vec.transpose(0, 2, 1).reshape(steps, LANES)


def _lane_record(sym_tile: np.ndarray, tab, x_init, seg: int = SEG_STEPS, lits=None):
    """Lane-stream record of one tile (FLAG_LANE_STREAMS).  sym_tile: uint8 [steps x 32] in tile order.

    Every lane is an ordinary scalar rANS stream (P:l.192 "each warp lane maintains its own rANS state"); instead
    of interleaving the lanes' 16-bit words in read order, each lane keeps its words to itself.  The tile is cut
    into segments of SEG_STEPS decode steps; a word belongs to the segment of the step after which the decoder
    reads it.  Inside a segment lanes 2p and 2p+1 share region p: lane 2p's words ascending from the region start,
    lane 2p+1's words descending from the region end (so 16 region sizes locate all 32 streams).

    record = [32 x u32 start states][per segment: u16 base, u16 total words, 16 x u8 (region words - base)]
             [segment 0 regions 0..15][segment 1 ...] zero-padded to 16 bytes.
    Returns (record bytes, number of payload words, staged bytes of the largest segment)."""
    steps = sym_tile.shape[0]
    assert steps % seg == 0, "lane-stream tiles must have a multiple of %d steps" % seg
    S = steps // seg
    states = np.zeros(LANES, dtype=np.uint64)
    seg_words = [[None] * LANES for _ in range(S)]
    for lane in range(LANES):
        col = np.ascontiguousarray(sym_tile[:, lane])
        if lits is not None:   # pair variant: escape literals ride in the lane's stream (codec.encode_scalar_lit)
            st, words, after = codec.encode_scalar_lit(col, tab, WORD_BITS, STATE_LO_LOG2, int(x_init[lane]), lits[lane])
            states[lane] = st
            used_prev = 0
            for sg in range(S):
                used = int(after[(sg + 1) * seg - 1])
                seg_words[sg][lane] = words[used_prev:used]
                used_prev = used
            assert used_prev == words.size
            continue
        st, words = codec.encode_scalar(col, tab, WORD_BITS, STATE_LO_LOG2, int(x_init[lane]))
        states[lane] = st
        used_prev = 0
        for sg in range(S):   # words the decoder has consumed after (sg+1)*seg steps
            _, _, used = codec.decode_scalar(st, words, (sg + 1) * seg, tab, WORD_BITS, STATE_LO_LOG2)
            seg_words[sg][lane] = words[used_prev:used]
            used_prev = used
        assert used_prev == words.size
    tables, body, n_words, max_seg = b"", b"", 0, 0
    for sg in range(S):
        sizes = [seg_words[sg][2 * p].size + seg_words[sg][2 * p + 1].size for p in range(LANES // 2)]
        base, total = min(sizes), sum(sizes)
        if max(sizes) - base > 255 or total > 0xFFFF:
            raise ValueError("lane-stream layout cannot represent this tile (region sizes spread over more than 255 words)")
        tables += struct.pack("<HH16B", base, total, *[z - base for z in sizes])
        for p in range(LANES // 2):
            body += seg_words[sg][2 * p].astype("<u2").tobytes() + seg_words[sg][2 * p + 1][::-1].astype("<u2").tobytes()
        n_words += total
        max_seg = max(max_seg, _align(15 + 2 * total) + 16)
    rec = states.astype("<u4").tobytes() + tables + body
    return rec + b"\0" * (_align(len(rec)) - len(rec)), n_words, max_seg


def _lane_record_decode(rec: np.ndarray, steps: int, tab, seg: int = SEG_STEPS, pair: bool = False):
    """Inverse of _lane_record: returns (symbols uint8 [steps x 32], end states[32]) and, for the pair variant,
    the literal of every nibble (uint16 [2*steps x 32], 0xFFFF = not an escape)."""
    S = steps // seg
    states = np.frombuffer(rec[:4 * LANES].tobytes(), dtype="<u4").astype(np.uint64)
    pos = 4 * LANES + 20 * S
    lanes = [[] for _ in range(LANES)]
    for sg in range(S):
        t = struct.unpack("<HH16B", rec[4 * LANES + 20 * sg:4 * LANES + 20 * sg + 20].tobytes())
        base, total, deltas = t[0], t[1], t[2:]
        if sum(base + d for d in deltas) != total:
            raise ValueError("corrupt lane-stream segment table")
        for p in range(LANES // 2):
            n = base + deltas[p]
            region = np.frombuffer(rec[pos:pos + 2 * n].tobytes(), dtype="<u2")
            lanes[2 * p].append((region, +1))
            lanes[2 * p + 1].append((region, -1))
            pos += 2 * n
    sym = np.zeros((steps, LANES), dtype=np.uint8)
    end = np.zeros(LANES, dtype=np.uint64)
    lit = np.full((2 * steps, LANES), 0xFFFF, dtype=np.uint16)
    # the split of a region between its two lanes is not stored: lane 2p decodes ascending, lane 2p+1 descending,
    # each taking exactly the words its own renormalisations (and escapes) ask for
    for lane in range(LANES):
        x = int(states[lane])
        out, lo = [], []
        for sg in range(S):
            region, d = lanes[lane][sg]
            words = region if d > 0 else region[::-1]
            if pair:
                o, l, x, _ = codec.decode_scalar_lit(x, words, seg, tab, WORD_BITS, STATE_LO_LOG2)
                lo.append(l)
            else:
                o, x, _ = codec.decode_scalar(x, words, seg, tab, WORD_BITS, STATE_LO_LOG2)
            out.append(o)
        sym[:, lane] = np.concatenate(out)
        if pair:
            lit[:, lane] = np.concatenate(lo)
        end[lane] = x
    return (sym, end, lit) if pair else (sym, end)


def encode(fmt: int, w: np.ndarray, k_in: int, tile_k: int = 0, flags: int = 0,
           scales: np.ndarray | None = None, zeros: np.ndarray | None = None,
           group_size: int = 0, w_scale: float = 1.0, tile_n: int = TILE_N):
    """Compress one weight matrix.  Returns (container bytes as np.uint8 array, stats dict).

    w: bf16 -> uint16 [n_out x k_in]; fp8/int8 -> (u)int8 [n_out x k_in]; int4 -> uint8 [n_out x k_in/2].
    scales/zeros: int8 -> fp16 [n_out]; int4 -> fp16 [n_out x k_in/group] each.
    """
    tile_k = tile_k or DEFAULT_TILE_K[fmt]
    pair = fmt == FMT_BF16_PAIR4
    if pair:
        assert (flags & FLAG_LANE_STREAMS) and tile_n == 32, "bf16 pair variant: lane streams on 32-row tiles only"
        coded, raw, exps, ctab = symbolise_pair(w)
    else:
        coded, raw = symbolise(fmt, w)
    n_out = coded.shape[0]
    assert n_out % STRIPE_N == 0 and k_in % tile_k == 0 and tile_n in (32, 128)
    if flags & FLAG_STATE_PAYLOAD:
        assert fmt in (FMT_BF16, FMT_BF16_PAIR4), "state payload carries raw-plane bytes: bf16 only"
    if flags & FLAG_LANE_STREAMS:
        assert tile_n == 32, "lane streams: 32-row tiles only"
    max_seg_bytes = 0
    wps = WEIGHTS_PER_SYMBOL[fmt]
    sym_cols = tile_k // wps
    KT = k_in // tile_k
    Q = STRIPE_N // tile_n                       # tiles per (stripe, k-tile) group; tile index = (stripe*KT + kt)*Q + q
    n_tiles = (n_out // STRIPE_N) * KT * Q
    L = 1 << STATE_LO_LOG2

    # P:l.167 "aggregate the weight statistics across the entire layer to construct a shared codebook"
    cnt = codec.histogram(coded)
    H = codec.entropy(cnt)
    f = codec.normalize(cnt, PROB_BITS)
    X = codec.cross_entropy(cnt, f, PROB_BITS)
    tab = codec.Table(f, PROB_BITS)

    rows, cols = tile_order(fmt, tile_k, tile_n)
    steps = rows.size // LANES
    records, raws, offsets = [], [], [0]
    state_bits = payload_bits = pad_bits = 0
    for stripe in range(n_out // STRIPE_N):
        for kt in range(KT):
            for q in range(Q):
                r0 = stripe * STRIPE_N + q * tile_n
                blk = coded[r0:r0 + tile_n, kt * sym_cols:(kt + 1) * sym_cols]
                sym = blk[rows, cols]
                x_init = np.full(LANES, L, dtype=np.uint64)
                lits = None
                if pair:   # one raw byte per WEIGHT (two per step): lane l = row l, vectors of 16 weights
                    rblk = raw[r0:r0 + tile_n, kt * tile_k:(kt + 1) * tile_k]
                    plane, payload = _raw_tile_pack(np.ascontiguousarray(rblk.T), flags)
                    raws.append(plane)
                    x_init = x_init + payload
                    eblk = exps[r0:r0 + tile_n, kt * tile_k:(kt + 1) * tile_k]
                    cw = np.zeros((tile_n, tile_k), dtype=np.uint8)
                    cw[:, 0::2], cw[:, 1::2] = blk & 15, blk >> 4
                    lits = [eblk[l][cw[l] == 15] for l in range(LANES)]       # in k order = step order, low nibble first
                elif raw is not None:
                    rblk = raw[r0:r0 + tile_n, kt * sym_cols:(kt + 1) * sym_cols]
                    plane, payload = _raw_tile_pack(rblk[rows, cols].reshape(steps, LANES), flags)
                    raws.append(plane)
                    x_init = x_init + payload
                if flags & FLAG_LANE_STREAMS:
                    rec, n_words, seg_bytes = _lane_record(sym.reshape(steps, LANES), tab, x_init, seg_steps(fmt), lits)
                    max_seg_bytes = max(max_seg_bytes, seg_bytes)
                    records.append(rec)
                    offsets.append(offsets[-1] + len(rec) // 16)
                    state_bits += 32 * LANES
                    payload_bits += 16 * n_words
                    pad_bits += 8 * (len(rec) - 4 * LANES - 2 * n_words)   # segment tables + padding
                    continue
                states, words = codec.tile_encode(sym, LANES, tab, WORD_BITS, STATE_LO_LOG2, x_init)
                rec = states.astype("<u4").tobytes() + words.astype("<u2").tobytes()
                pad = _align(len(rec)) - len(rec)
                records.append(rec + b"\0" * pad)
                offsets.append(offsets[-1] + (len(rec) + pad) // 16)
                state_bits += 32 * LANES
                payload_bits += 16 * words.size
                pad_bits += 8 * pad

    rec_bytes = b"".join(records)
    raw_bytes = np.concatenate(raws).tobytes() if raws else b""
    side = b""
    if fmt == FMT_INT8:
        side = np.ascontiguousarray(scales, dtype=np.float16).tobytes()
    elif fmt == FMT_INT4_AWQ:
        s = np.ascontiguousarray(scales, dtype=np.float16)           # [n_out x groups]
        z = np.ascontiguousarray(zeros, dtype=np.float16)
        sz = np.stack([s.T, z.T], axis=-1)                           # [groups x n_out x (s, z)]
        side = np.ascontiguousarray(sz).tobytes()

    off_freq = HEADER_BYTES
    off_offsets = _align(off_freq + 512)
    off_records = _align(off_offsets + 4 * (n_tiles + 1))
    off_raw = _align(off_records + len(rec_bytes))
    off_scales = _align(off_raw + len(raw_bytes))
    total = _align(off_scales + len(side))
    off_codes = 0
    if pair:   # the 16-byte exponent code table sits where no other format has a section (header field off_zeros)
        off_codes = off_scales
        total = _align(off_codes + 16)
    total = max(total, _align(off_records + len(rec_bytes) + TAIL_BYTES))   # tail rule
    hdr = Header(fmt, n_out, k_in, tile_n, tile_k, LANES, PROB_BITS, WORD_BITS, STATE_LO_LOG2, group_size, flags,
                 n_tiles, float(w_scale), off_freq, off_offsets, off_records, off_raw if raw_bytes else 0,
                 off_scales if side else 0, off_codes, total, max_seg_bytes)
    buf = np.zeros(total, dtype=np.uint8)
    buf[:HEADER_BYTES] = np.frombuffer(hdr.pack(), dtype=np.uint8)
    buf[off_freq:off_freq + 512] = np.frombuffer(f.astype("<u2").tobytes(), dtype=np.uint8)
    buf[off_offsets:off_offsets + 4 * (n_tiles + 1)] = np.frombuffer(np.asarray(offsets, dtype="<u4").tobytes(), dtype=np.uint8)
    buf[off_records:off_records + len(rec_bytes)] = np.frombuffer(rec_bytes, dtype=np.uint8)
    if raw_bytes:
        buf[off_raw:off_raw + len(raw_bytes)] = np.frombuffer(raw_bytes, dtype=np.uint8)
    if side:
        buf[off_scales:off_scales + len(side)] = np.frombuffer(side, dtype=np.uint8)
    if pair:
        buf[off_codes:off_codes + 16] = ctab

    n_weights = n_out * k_in
    H_raw = codec.entropy(codec.histogram(raw)) if raw is not None else 0.0
    stats = dict(n_weights=n_weights, payload_bits=payload_bits, state_bits=state_bits, pad_bits=pad_bits,
                 offset_table_bits=32 * (n_tiles + 1), freq_table_bits=512 * 8, raw_bits=8 * len(raw_bytes),
                 side_bits=8 * len(side), entropy_bits_per_symbol=H, xent_bits_per_symbol=X,
                 raw_entropy_bits_per_symbol=H_raw,
                 # reading A2/A22: H_sym per weight = sum over planes; scales/zeros excluded from both sides
                 h_sym_bits_per_weight=H / wps + H_raw,
                 bits_per_weight=8.0 * (total - len(side)) / n_weights,
                 total_bytes=total)
    return buf, stats


def decode(buf: np.ndarray):
    """Decompress a container (from either encoder).  Returns (header, w, side) with w in the
    caller's original dtype/packing (bf16 -> uint16 bit patterns)."""
    buf = np.ascontiguousarray(buf, dtype=np.uint8)
    h = Header.unpack(buf)
    fmt, tile_k, tile_n = h.fmt, h.tile_k, h.tile_n
    if tile_n not in (32, 128):
        raise ValueError("unsupported tile_n %d" % tile_n)
    Q = STRIPE_N // tile_n
    wps = WEIGHTS_PER_SYMBOL[fmt]
    sym_cols = tile_k // wps
    KT = h.k_in // tile_k
    f = np.frombuffer(buf[h.off_freq:h.off_freq + 512].tobytes(), dtype="<u2").astype(np.uint32)
    tab = codec.Table(f, h.prob_bits)
    offsets = np.frombuffer(buf[h.off_offsets:h.off_offsets + 4 * (h.n_tiles + 1)].tobytes(), dtype="<u4").astype(np.int64)
    rows, cols = tile_order(fmt, tile_k, tile_n)
    n_sym = rows.size
    steps = n_sym // LANES
    L = 1 << h.state_lo_log2
    coded = np.zeros((h.n_out, h.k_in // wps), dtype=np.uint8)
    pair = fmt == FMT_BF16_PAIR4
    raw = np.zeros_like(coded) if fmt == FMT_BF16 else (np.zeros((h.n_out, h.k_in), dtype=np.uint8) if pair else None)
    lit_all = np.full((h.n_out, h.k_in), 0xFFFF, dtype=np.uint16) if pair else None
    rtb = raw_tile_bytes(tile_k, h.flags, tile_n)
    t = 0
    for stripe in range(h.n_out // STRIPE_N):
        for kt, q in ((kt, q) for kt in range(KT) for q in range(Q)):
            r0 = stripe * STRIPE_N + q * tile_n
            a = h.off_records + 16 * int(offsets[t])
            e = h.off_records + 16 * int(offsets[t + 1])
            if pair:
                sym, end, lit = _lane_record_decode(buf[a:e], steps, tab, seg_steps(fmt), True)
                sym = sym.reshape(-1)
                used = (e - a - 4 * LANES) // 2
                lit_all[r0:r0 + tile_n, kt * tile_k:(kt + 1) * tile_k] = lit.T
            elif h.flags & FLAG_LANE_STREAMS:
                sym, end = _lane_record_decode(buf[a:e], steps, tab, seg_steps(fmt))
                sym = sym.reshape(-1)
                used = (e - a - 4 * LANES) // 2
            else:
                states = np.frombuffer(buf[a:a + 4 * LANES].tobytes(), dtype="<u4").astype(np.uint64)
                words = np.frombuffer(buf[a + 4 * LANES:e].tobytes(), dtype="<u2")
                sym, end, used = codec.tile_decode(states, words, n_sym, LANES, tab, h.word_bits, h.state_lo_log2)
            payload = end - np.uint64(L)
            if h.flags & FLAG_STATE_PAYLOAD:
                if np.any(end < L) or np.any(payload > 0xFFFF):
                    raise ValueError("corrupt tile %d: end state out of range" % t)
            elif np.any(end != L):
                raise ValueError("corrupt tile %d: end state != L" % t)
            if (e - a - 4 * LANES) // 2 - used not in range(0, 8):
                raise ValueError("corrupt tile %d: %d words stored, %d used" % (t, (e - a - 128) // 2, used))
            blk = np.zeros((tile_n, sym_cols), dtype=np.uint8)
            blk[rows, cols] = sym
            coded[r0:r0 + tile_n, kt * sym_cols:(kt + 1) * sym_cols] = blk
            if pair:
                plane = buf[h.off_raw + t * rtb:h.off_raw + (t + 1) * rtb]
                raw[r0:r0 + tile_n, kt * tile_k:(kt + 1) * tile_k] = _raw_tile_unpack(plane, tile_k, h.flags, payload).T
            elif raw is not None:
                plane = buf[h.off_raw + t * rtb:h.off_raw + (t + 1) * rtb]
                rl = _raw_tile_unpack(plane, steps, h.flags, payload)
                rblk = np.zeros((tile_n, sym_cols), dtype=np.uint8)
                rblk[rows, cols] = rl.reshape(-1)
                raw[r0:r0 + tile_n, kt * sym_cols:(kt + 1) * sym_cols] = rblk
            t += 1
    if pair:
        ctab = buf[h.off_zeros:h.off_zeros + 16]
        cw = np.zeros((h.n_out, h.k_in), dtype=np.uint8)
        cw[:, 0::2], cw[:, 1::2] = coded & 15, coded >> 4
        if np.any((cw == 15) != (lit_all != 0xFFFF)) or np.any(lit_all[cw == 15] > 0xFF):
            raise ValueError("corrupt container: escape literals do not match the escape codes")
        exps = np.where(cw == 15, lit_all.astype(np.uint8), ctab[np.minimum(cw, 14)])
        w = desymbolise(FMT_BF16, exps, raw)
    else:
        w = desymbolise(fmt, coded, raw)
    side = {}
    if fmt == FMT_INT8:
        side["scales"] = np.frombuffer(buf[h.off_scales:h.off_scales + 2 * h.n_out].tobytes(), dtype=np.float16)
    elif fmt == FMT_INT4_AWQ:
        groups = h.k_in // h.group_size
        sz = np.frombuffer(buf[h.off_scales:h.off_scales + 4 * groups * h.n_out].tobytes(), dtype=np.float16)
        sz = sz.reshape(groups, h.n_out, 2)
        side["scales"] = np.ascontiguousarray(sz[:, :, 0].T)
        side["zeros"] = np.ascontiguousarray(sz[:, :, 1].T)
    return h, w, side


def metadata_bytes_eq3(n_tiles: int, b: int = 12) -> int:
    """Eq.3 (P:l.440): 4 B per tile offset + 2^b * 4 B shared codebook."""
    return 4 * n_tiles + (1 << b) * 4
