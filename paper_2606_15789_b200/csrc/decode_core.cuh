// Warp-cooperative rANS tile decoder (Alg V.2, P:l.260-287), sm_100a.
//
// One warp lane owns one of the 32 interleaved streams of a tile (P:l.192 "each warp lane maintains
// its own rANS state").  Per step and lane:  slot = x & 4095;  e = T[slot] (shared-memory table,
// P:l.271);  x = f*(x>>12) + bias;  if x < 2^16: x = x<<16 | next word.  The words of a tile are
// interleaved in decoder read order, so the renormalising lanes of a step read CONSECUTIVE 16-bit
// words (P:l.256 "renormalization loads are naturally coalesced"): ballot + popc prefix picks the word.
//
// A decode step is a dependent chain (LDS table -> IMAD -> renormalise: 74 clk for one lane-stream chain alone on an
// SM, 86 clk for two interleaved; more with ballot / prefix count of the interleaved-word layout), so
// throughput comes from independent chains in flight: a warp decodes J tiles at once, their steps
// interleaved instruction by instruction (J = 2 for 32-row tiles), and many such warps share an SM.
//
// The compressed words stream HBM -> shared memory through a 2 KiB ring per stream (+ a 512-byte
// mirror of its first block, so that the 8 steps between two upkeeps address the ring linearly)
// with 16-byte cp.async: 32 lanes x 16 B = one 512-byte block per fill.
//
// Table entry (4 B, Eq.3's "2^b x 4 B", P:l.440):  sym[7:0] | f[19:8] | bias[31:20].
#pragma once
#include <cuda_fp16.h>
#include <stdint.h>
#include <type_traits>
#include "anslin_internal.h"

namespace anslin {

constexpr uint32_t kRingBytes = 2048;    // per stream
constexpr uint32_t kFillBytes = 512;     // 32 lanes x 16 B per fill
constexpr uint32_t kMirrorBytes = 512;   // copy of ring block 0 behind the ring
constexpr uint32_t kStreamSmem = kRingBytes + kMirrorBytes;
// The ring reads ahead of the record it decodes: the container guarantees this many readable bytes
// after the records section (tail rule), so fills need no bounds check.
static_assert(2 * kRingBytes <= uint32_t(kTailBytes), "ring read-ahead must fit the container tail rule");

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}
__device__ __forceinline__ void sts128(uint32_t a, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint32_t lds32v(uint32_t a) {
  uint32_t v;
  asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }
__device__ __forceinline__ uint4 ldg128_stream(const void *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// Expand the 256 x u16 frequency table of the container into the 4096-entry slot table in shared
// memory (Alg V.1 l.6 "Copy global decode table T into shared memory", P:l.212).  All threads of
// the CTA must call; `cum` is 257 u32 of scratch.  Ends with __syncthreads().
// Split in two so that a caller can have the table's HBM round trip in flight under other loads: lane l of warp 0 holds
// frequencies 8l .. 8l+7 (one 16-byte load).
__device__ __forceinline__ uint4 slot_table_load(const uint16_t *freq_g) {
  uint4 fr = make_uint4(0, 0, 0, 0);
  if (threadIdx.x < 32) fr = *reinterpret_cast<const uint4 *>(freq_g + threadIdx.x * 8);   // off_freq is 16-byte aligned
  return fr;
}
__device__ __forceinline__ void build_slot_table(uint32_t *tab, uint32_t *cum, const uint4 fr) {
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
  if (warp == 0) {  // exclusive prefix sum of 256 frequencies: 8 per lane + warp scan
    const uint32_t w[4] = {fr.x, fr.y, fr.z, fr.w};
    uint32_t f[8], s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { f[i] = (w[i >> 1] >> (16 * (i & 1))) & 0xFFFFu; s += f[i]; }
    uint32_t inc = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
      if (lane >= d) inc += o;
    }
    uint32_t run = inc - s;
#pragma unroll
    for (int i = 0; i < 8; ++i) { cum[lane * 8 + i] = run; run += f[i]; }
    if (lane == 31) cum[256] = run;
  }
  __syncthreads();
  for (int s = warp; s < 256; s += nwarp) {
    const uint32_t c0 = cum[s], f = cum[s + 1] - c0;
    for (uint32_t k = lane; k < f; k += 32) tab[c0 + k] = uint32_t(s) | (k << 8) | (f << 20);
  }
  __syncthreads();
}
__device__ __forceinline__ void build_slot_table(uint32_t *tab, uint32_t *cum, const uint16_t *freq_g) {
  build_slot_table(tab, cum, slot_table_load(freq_g));
}

// One lane's view of one tile's compressed stream.
struct Stream {
  uint32_t x;      // this lane's rANS state
  uint32_t pa;     // shared address of the next unread word (warp uniform; may run into the mirror)
  uint32_t bal;    // (bytes whose fill has been issued minus bytes consumed) + pa, as of the last upkeep
  uint32_t fa;     // shared address of this lane's 16-byte slice of the next fill block
  const uint8_t *src;  // this lane's next fill source = words + issued + 16*lane
};

// rec = start of the tile record in HBM (16-byte aligned); ring = shared address of kStreamSmem bytes.
// The caller must have drained earlier cp.async groups into this ring (stream_drain) first.
__device__ __forceinline__ void stream_open(Stream &s, const uint8_t *rec, uint32_t ring, int lane) {
  s.x = reinterpret_cast<const uint32_t *>(rec)[lane];
  const uint8_t *src = rec + 4 * kLanes + 16 * lane;
  const uint32_t fa = ring + 16u * uint32_t(lane);
#pragma unroll
  for (uint32_t b = 0; b < 3; ++b)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(fa + b * kFillBytes), "l"(src + b * kFillBytes) : "memory");
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(fa + kRingBytes), "l"(src) : "memory");  // mirror of block 0
  cp_async_commit();
  s.src = src + 3 * kFillBytes;
  s.fa = fa + 3 * kFillBytes;
  s.pa = ring;
  s.bal = 3 * kFillBytes + ring;
}
__device__ __forceinline__ void stream_drain() {
  cp_async_wait_all();
  __syncwarp();
}

// Ring upkeep of J streams before their next EIGHT decode steps (which consume at most 448 B each:
// a lane renormalises in at most 7 of 8 steps).  Policy: refill one 512-byte block whenever the
// issued-but-unread lead has dropped to <= 1024 B.  Invariants on entry: lead >= 641 > 448 and every
// fill but the one issued by the PREVIOUS upkeep has landed; the single wait_group 1 below (after
// this upkeep's commit) retires that one, so all `lead` bytes are readable when the steps start.
// A fill overwrites ring bytes [issued - 2048, issued - 1536) < consumed.  The mirror makes
// addresses linear for 512 B past the ring end; pa wraps here, once per 8 steps.
// ring0 = shared address of stream 0's ring; stream j's ring follows at j * kStreamSmem.
template <int J>
__device__ __forceinline__ void stream_upkeep8(Stream (&s)[J], uint32_t ring0, int lane) {
#pragma unroll
  for (int j = 0; j < J; ++j) {
    Stream &t = s[j];
    const uint32_t lim = ring0 + uint32_t(j) * kStreamSmem + kRingBytes;
    const uint32_t lead = t.bal - t.pa;
    if (t.pa >= lim) t.pa -= kRingBytes;
    t.bal = lead + t.pa;
    if (lead <= 1024u) {
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(t.fa), "l"(t.src) : "memory");
      if (t.fa < lim - kRingBytes + kFillBytes)   // block 0 also feeds the mirror
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(t.fa + kRingBytes), "l"(t.src) : "memory");
      t.fa += kFillBytes;
      if (t.fa >= lim) t.fa -= kRingBytes;
      t.src += kFillBytes;
      t.bal += kFillBytes;
    }
  }
  cp_async_commit();
  cp_async_wait_1();
  __syncwarp();
}

// x' = f * (x >> b) + (slot - c) (Alg V.2 l.7, P:l.276) from the table entry e = sym | (slot - c) << 8 | f << 20.  Two shifts
// and no mask: e >> 8 = f << 12 | (slot - c) carries f * 2^12 too much, which the multiplicand (x >> 12) - 2^12 takes back
// (all modulo 2^32; the result is < 2^32 as in the plain form).
__device__ __forceinline__ uint32_t state_update(uint32_t x, uint32_t e) {
  return (e >> 20) * ((x >> kProbBits) - (1u << kProbBits)) + (e >> 8);
}
// One decode step of Alg V.2 for all 32 lanes of one stream; returns the table entry (symbol in bits 7:0).
__device__ __forceinline__ uint32_t decode_step(Stream &s, uint32_t tab_s, uint32_t lt) {
  uint32_t ea, e;
  asm("mul.lo.u32 %0, %1, 4;" : "=r"(ea) : "r"(s.x));          // shift on the FMA pipe (IMAD.SHL), mask on the ALU,
  asm("and.b32 %0, %0, 0x3FFC;" : "+r"(ea));                   // table base folded into the load's address operand
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(e) : "r"(ea + tab_s));
  uint32_t xn = state_update(s.x, e);
  // renormalisation: the lanes with x < 2^16 read consecutive words, x = (x << 16) | word
  asm volatile(
      "{\n\t.reg .pred p;\n\t.reg .u16 h;\n\t.reg .u32 w, m, r, a;\n\t"
      "setp.lt.u32 p, %0, 65536;\n\t"
      "vote.sync.ballot.b32 m, p, 0xffffffff;\n\t"
      "and.b32 r, m, %2;\n\t"
      "popc.b32 r, r;\n\t"
      "mad.lo.u32 a, r, 2, %1;\n\t"
      "ld.shared.u16 h, [a];\n\t"      // every lane loads (same 64-byte window): keeps w defined on all paths
      "cvt.u32.u16 w, h;\n\t"
      "@p mad.lo.u32 %0, %0, 65536, w;\n\t"
      "popc.b32 m, m;\n\t"
      "mad.lo.u32 %1, m, 2, %1;\n\t}"
      : "+r"(xn), "+r"(s.pa)
      : "r"(lt)
      : "memory");
  s.x = xn;
  return e;
}

// ---- lane-stream layout (ANSLIN_FLAG_LANE_STREAMS): every lane reads its own word stream ----------------
// The record is cut into segments of seg_steps_of(format) decode steps; a segment's words are staged whole in shared
// memory, lanes 2p and 2p+1 sharing region p (lane 2p walks up from its start, lane 2p+1 down from its end).
// No ballot, no prefix count, no ring upkeep: a step renormalises with a predicated load at the lane's cursor.
struct LaneStream {
  uint32_t x;          // this lane's rANS state
  uint32_t ptr;        // shared address of this lane's next word
  uint32_t w;          // that word, loaded ahead: a renormalisation takes it from the register, then fetches the next
                       // one, so the shared-memory latency of the word is off the state's dependency chain
  uint32_t goff;       // byte offset, from the record start, of the next segment's words
  const uint8_t *rec;  // record start in HBM
};
__device__ __forceinline__ void lane_open(LaneStream &s, const uint8_t *rec, int segments, int lane) {
  s.x = reinterpret_cast<const uint32_t *>(rec)[lane];
  s.rec = rec;
  s.goff = 4 * kLanes + uint32_t(kSegTableBytes) * uint32_t(segments);
  s.w = 0;
  s.ptr = 0;
}
// Stage segment `seg` of J records into their buffers (stream j's at buf0 + j * bufbytes) and point every lane at
// its stream.  All lanes have finished reading the previous segments (program order + the __syncwarp in
// stream_drain).  The segment tables and the words are fetched together: when the buffer is no larger than the
// container's tail rule allows to over-read, the whole buffer is copied from the segment start without waiting
// for the table to say how many words there are.
struct NoExtraCopies { __device__ __forceinline__ void operator()() const {} };
// extra(): further cp.async copies of the caller, issued into the same group as the segment's (one wait for both)
template <int J, class Extra = NoExtraCopies>
__device__ __forceinline__ void lane_open_segments(LaneStream (&s)[J], uint32_t buf0, uint32_t bufbytes, int seg, int lane,
                                                   const Extra &extra = Extra()) {
  stream_drain();
  const bool spec = bufbytes <= uint32_t(kTailBytes);
  uint32_t hdr[J], delta[J];
#pragma unroll
  for (int j = 0; j < J; ++j) {
    const uint8_t *te = s[j].rec + 4 * kLanes + kSegTableBytes * seg;
    hdr[j] = *reinterpret_cast<const uint32_t *>(te);   // u16 base | u16 total words
    delta[j] = lane < kLanes / 2 ? uint32_t(te[4 + lane]) : 0u;
    if (spec) {
      const uint32_t skew = s[j].goff & 15u;
      const uint8_t *src = s[j].rec + (s[j].goff - skew);
      for (uint32_t o = 16u * uint32_t(lane); o < bufbytes; o += kFillBytes)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(buf0 + uint32_t(j) * bufbytes + o), "l"(src + o) : "memory");
    }
  }
#pragma unroll
  for (int j = 0; j < J; ++j) {
    const uint32_t base = hdr[j] & 0xFFFFu, total = hdr[j] >> 16, buf = buf0 + uint32_t(j) * bufbytes;
    const uint32_t size = lane < kLanes / 2 ? base + delta[j] : 0u;   // words of region `lane`
    uint32_t end = size;
#pragma unroll
    for (int d = 1; d < kLanes / 2; d <<= 1) {
      const uint32_t o = __shfl_up_sync(0xffffffffu, end, d);
      if (lane >= d) end += o;
    }
    const uint32_t start = end - size;
    const uint32_t start_p = __shfl_sync(0xffffffffu, start, lane >> 1), end_p = __shfl_sync(0xffffffffu, end, lane >> 1);
    const uint32_t skew = s[j].goff & 15u;
    if (!spec) {
      const uint8_t *src = s[j].rec + (s[j].goff - skew);
      const uint32_t nbytes = min((skew + 2u * total + 15u) & ~15u, bufbytes);   // a damaged table cannot overrun the buffer
      for (uint32_t o = 16u * uint32_t(lane); o < nbytes; o += kFillBytes)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(buf + o), "l"(src + o) : "memory");
    }
    // the cursor is clamped into the staged buffer: a damaged table (anslin_open cannot check a container whose records
    // never were on the host) yields wrong weights, never an address outside the buffer
    s[j].ptr = buf + skew + 2u * min((lane & 1) ? end_p - 1u : start_p, (bufbytes - skew) / 2u - 1u);
    s[j].goff += 2u * total;
  }
  extra();
  cp_async_commit();
  stream_drain();
  // look-ahead word (a lane without words in this segment reads a neighbour's or stale bytes: never used)
#pragma unroll
  for (int j = 0; j < J; ++j) asm volatile("ld.shared.u16 %0, [%1];" : "=r"(s[j].w) : "r"(s[j].ptr) : "memory");
}
// One decode step of Alg V.2 for all 32 lanes of one lane-stream tile; dir = +2 (even lanes) / -2 (odd lanes).
__device__ __forceinline__ uint32_t lane_step(LaneStream &s, uint32_t tab_s, uint32_t dir) {
  uint32_t ea, e;
  asm("mul.lo.u32 %0, %1, 4;" : "=r"(ea) : "r"(s.x));          // shift on the FMA pipe (IMAD.SHL), mask on the ALU,
  asm("and.b32 %0, %0, 0x3FFC;" : "+r"(ea));                   // table base folded into the load's address operand
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(e) : "r"(ea + tab_s));
  uint32_t xn = state_update(s.x, e);
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.lt.u32 p, %0, 65536;\n\t"
      "@p mad.lo.u32 %0, %0, 65536, %2;\n\t"
      "@p add.u32 %1, %1, %3;\n\t"
      "@p ld.shared.u16 %2, [%1];\n\t}"
      : "+r"(xn), "+r"(s.ptr), "+r"(s.w)
      : "r"(dir)
      : "memory");
  s.x = xn;
  return e;
}

// Two lane-stream tiles, one step each, written so that the in-order issue overlaps the two dependent chains: both
// table loads first, then both state updates, then both merges with the look-ahead words, then the predicated
// loads of the next look-ahead words.
__device__ __forceinline__ void lane_step2(LaneStream &s0, LaneStream &s1, uint32_t tab_s, uint32_t dir, uint32_t &e0, uint32_t &e1) {
  uint32_t a0, a1;
  asm("mul.lo.u32 %0, %1, 4;" : "=r"(a0) : "r"(s0.x));
  asm("mul.lo.u32 %0, %1, 4;" : "=r"(a1) : "r"(s1.x));
#ifdef ANSLIN_SKEL_NOCONFLICT   // timing experiment only (wrong results): the table gather without bank conflicts
  { const uint32_t l4 = (threadIdx.x & 31u) << 2;
    asm("lop3.b32 %0, %0, 0x3F80, %1, 0xEA;" : "+r"(a0) : "r"(l4));
    asm("lop3.b32 %0, %0, 0x3F80, %1, 0xEA;" : "+r"(a1) : "r"(l4)); }
#else
  asm("and.b32 %0, %0, 0x3FFC;" : "+r"(a0));
  asm("and.b32 %0, %0, 0x3FFC;" : "+r"(a1));
#endif
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(e0) : "r"(a0 + tab_s));
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(e1) : "r"(a1 + tab_s));
  uint32_t x0 = state_update(s0.x, e0);
  uint32_t x1 = state_update(s1.x, e1);
  asm volatile(
      "{\n\t.reg .pred p, q;\n\t"
      "setp.lt.u32 p, %0, 65536;\n\t"
      "setp.lt.u32 q, %3, 65536;\n\t"
      "@p mad.lo.u32 %0, %0, 65536, %2;\n\t"
      "@q mad.lo.u32 %3, %3, 65536, %5;\n\t"
      "@p add.u32 %1, %1, %6;\n\t"
      "@q add.u32 %4, %4, %6;\n\t"
#ifndef ANSLIN_SKEL_NOWORDLOAD   // timing experiment only (wrong results): no look-ahead word loads
      "@p ld.shared.u16 %2, [%1];\n\t"
      "@q ld.shared.u16 %5, [%4];\n\t"
#endif
      "}"
      : "+r"(x0), "+r"(s0.ptr), "+r"(s0.w), "+r"(x1), "+r"(s1.ptr), "+r"(s1.w)
      : "r"(dir)
      : "memory");
  s0.x = x0;
  s1.x = x1;
}

// The two word layouts as policies of decode_unit.
struct InterleavedWords {
  using S = Stream;
  template <int J> static __device__ __forceinline__ void upkeep8(S (&s)[J], uint32_t ring0, int lane) { stream_upkeep8<J>(s, ring0, lane); }
  static __device__ __forceinline__ uint32_t step(S &s, uint32_t tab, uint32_t lt) { return decode_step(s, tab, lt); }
  template <int J> static __device__ __forceinline__ void steps(S (&s)[J], uint32_t tab, uint32_t lt, uint32_t (&e)[J]) {
#pragma unroll
    for (int j = 0; j < J; ++j) e[j] = decode_step(s[j], tab, lt);
  }
};
struct LaneWords {
  using S = LaneStream;
  template <int J> static __device__ __forceinline__ void upkeep8(S (&)[J], uint32_t, int) {}
  static __device__ __forceinline__ uint32_t step(S &s, uint32_t tab, uint32_t dir) { return lane_step(s, tab, dir); }
  // one step of each of the J streams
  template <int J> static __device__ __forceinline__ void steps(S (&s)[J], uint32_t tab, uint32_t dir, uint32_t (&e)[J]) {
    if constexpr (J == 2) {
      lane_step2(s[0], s[1], tab, dir, e[0], e[1]);
    } else {
#pragma unroll
      for (int j = 0; j < J; ++j) e[j] = lane_step(s[j], tab, dir);
    }
  }
};

// Insert the symbol byte of table entry e at byte position `pos` of acc.
template <int pos>
__device__ __forceinline__ uint32_t put_sym(uint32_t acc, uint32_t e) {
  return __byte_perm(acc, e, (0x3210 & ~(0xF << (4 * pos))) | (4 << (4 * pos)));
}
// Four decode steps of each of the J streams, interleaved -> four symbol bytes per stream.
template <class POL, int J>
__device__ __forceinline__ void decode4(typename POL::S (&s)[J], uint32_t (&q)[J], uint32_t tab, uint32_t aux) {
  uint32_t e[J];
  POL::template steps<J>(s, tab, aux, e);
#pragma unroll
  for (int j = 0; j < J; ++j) q[j] = put_sym<0>(0u, e[j]);
  POL::template steps<J>(s, tab, aux, e);
#pragma unroll
  for (int j = 0; j < J; ++j) q[j] = put_sym<1>(q[j], e[j]);
  POL::template steps<J>(s, tab, aux, e);
#pragma unroll
  for (int j = 0; j < J; ++j) q[j] = put_sym<2>(q[j], e[j]);
  POL::template steps<J>(s, tab, aux, e);
#pragma unroll
  for (int j = 0; j < J; ++j) q[j] = put_sym<3>(q[j], e[j]);
}

// bf16: two decode steps + two raw bytes (R = mantissa<<1 | sign, bytes 2k', 2k'+1 of Rw) -> two bf16 values.
// p = [R_a, E_a, R_b, E_b] (two PRMTs straight from the table entries), then each 16-bit (E<<8 | R) is rotated
// right by one bit: shift, shift, one bit-select.
template <int KP>
__device__ __forceinline__ uint32_t bf16_pair(uint32_t Rw, uint32_t e_a, uint32_t e_b) {
  const uint32_t t = __byte_perm(Rw, e_a, KP == 0 ? 0x0140 : 0x0342);   // [R_a, E_a, R_b, -]
  const uint32_t p = __byte_perm(t, e_b, 0x4210);                        // [R_a, E_a, R_b, E_b]
  uint32_t o;
  asm("lop3.b32 %0, %1, %2, 0x7FFF7FFF, 0xE4;" : "=r"(o) : "r"(p >> 1), "r"(p << 15));   // (a & c) | (b & ~c)
  return o;
}
// Eight decode steps of each of the J streams, interleaved, merged with 8 raw bytes (R0, R1) -> one 16-byte chunk each.
template <class POL, int J>
__device__ __forceinline__ void decode8_bf16(typename POL::S (&s)[J], uint32_t tab, uint32_t aux, const uint32_t (&R0)[J],
                                             const uint32_t (&R1)[J], uint4 (&out)[J]) {
  uint32_t ea[J], eb[J];
#define ANSLIN_PAIR(KP, RW, DST)                                              \
  POL::template steps<J>(s, tab, aux, ea);                                    \
  POL::template steps<J>(s, tab, aux, eb);                                    \
  _Pragma("unroll") for (int j = 0; j < J; ++j) out[j].DST = bf16_pair<KP>(RW[j], ea[j], eb[j]);
  ANSLIN_PAIR(0, R0, x)
  ANSLIN_PAIR(1, R0, y)
  ANSLIN_PAIR(0, R1, z)
  ANSLIN_PAIR(1, R1, w)
#undef ANSLIN_PAIR
}

// int4 (AWQ-style): one packed byte (low nibble = even k) -> two fp16 weights (q - z) * s.
// 0x6400 | q is the fp16 number 1024 + q, so (1024+q) - (1024+z) is exact and the product rounds once.
__device__ __forceinline__ uint32_t awq_dequant2(uint32_t byte, __half2 zoff, __half2 sc) {
  const uint32_t v = (byte & 0x0Fu) | ((byte & 0xF0u) << 12) | 0x64006400u;
  __half2 h = *reinterpret_cast<const __half2 *>(&v);
  h = __hmul2(__hsub2(h, zoff), sc);
  return *reinterpret_cast<const uint32_t *>(&h);
}

// The same for four packed bytes at once: the nibbles are split once, then every byte costs one PRMT (a selector nibble with
// bit 3 set replicates the sign bit of the chosen byte, and a nibble byte is <= 0x0F: zero) and one OR before the two half2 ops.
__device__ __forceinline__ void awq_dequant8(uint32_t Bq, __half2 zoff, __half2 sc, uint32_t &o0, uint32_t &o1, uint32_t &o2, uint32_t &o3) {
  const uint32_t lo = Bq & 0x0F0F0F0Fu, hi = (Bq >> 4) & 0x0F0F0F0Fu;
  uint32_t v0, v1, v2, v3;   // (PTX prmt: __byte_perm does not pass the selector's replicate bits through)
  asm("prmt.b32 %0, %1, %2, 0x8480;" : "=r"(v0) : "r"(lo), "r"(hi));
  asm("prmt.b32 %0, %1, %2, 0x9591;" : "=r"(v1) : "r"(lo), "r"(hi));
  asm("prmt.b32 %0, %1, %2, 0xA6A2;" : "=r"(v2) : "r"(lo), "r"(hi));
  asm("prmt.b32 %0, %1, %2, 0xB7B3;" : "=r"(v3) : "r"(lo), "r"(hi));
  v0 |= 0x64006400u; v1 |= 0x64006400u; v2 |= 0x64006400u; v3 |= 0x64006400u;
  __half2 h0 = __hmul2(__hsub2(*reinterpret_cast<const __half2 *>(&v0), zoff), sc), h1 = __hmul2(__hsub2(*reinterpret_cast<const __half2 *>(&v1), zoff), sc);
  __half2 h2 = __hmul2(__hsub2(*reinterpret_cast<const __half2 *>(&v2), zoff), sc), h3 = __hmul2(__hsub2(*reinterpret_cast<const __half2 *>(&v3), zoff), sc);
  o0 = *reinterpret_cast<const uint32_t *>(&h0); o1 = *reinterpret_cast<const uint32_t *>(&h1);
  o2 = *reinterpret_cast<const uint32_t *>(&h2); o3 = *reinterpret_cast<const uint32_t *>(&h3);
}

// fp4-e2m1 (s.ee.m: 0, 0.5, 1, 1.5, 2, 3, 4, 6) -> the e4m3 byte of the same value, four codes at a time: the four
// nibbles of sel[15:0] pick their magnitude byte from an 8-entry table held in two registers (PRMT), the sign
// nibble-bit picks 0x00 / 0x80.  `mag` = codes & 0x7777..., `sgn` = (codes >> 3) & 0x1111... (upper 16 bits ignored).
__device__ __forceinline__ uint32_t e2m1x4_to_e4m3(uint32_t mag, uint32_t sgn) {
  return __byte_perm(0x3C383000u, 0x4C484440u, mag) | __byte_perm(0x00008000u, 0u, sgn);
}
// four packed bytes (8 codes, low nibble first) -> two words of e4m3 operand bytes
__device__ __forceinline__ void e2m1x8_to_e4m3(uint32_t b, uint32_t &lo, uint32_t &hi) {
  const uint32_t mag = b & 0x77777777u, sgn = (b >> 3) & 0x11111111u;
  lo = e2m1x4_to_e4m3(mag, sgn);
  hi = e2m1x4_to_e4m3(mag >> 16, sgn >> 16);
}

// ---- bf16 pair variant (ANSLIN_FMT_BF16_PAIR4): a coded byte holds the 4-bit exponent codes of two K-adjacent weights ----
struct PairLut { uint32_t t0, t1, t2, t3; };   // code -> exponent byte for codes 0..15 (the container's 16-byte code table)
// q = 4 coded bytes = the codes of 8 weights (nibble n = weight n) -> their exponent bytes, weights 0..3 in lo, 4..7 in hi.
// Two 8-entry PRMT look-ups per four codes, chosen per byte by the code's top bit (PRMT in sign-replication mode).
__device__ __forceinline__ void pair_exps(uint32_t q, const PairLut &L, uint32_t &lo, uint32_t &hi) {
  const uint32_t m = q & 0x77777777u, q4 = q << 4;
  const uint32_t a0 = __byte_perm(L.t0, L.t1, m), b0 = __byte_perm(L.t2, L.t3, m);
  const uint32_t a1 = __byte_perm(L.t0, L.t1, m >> 16), b1 = __byte_perm(L.t2, L.t3, m >> 16);
  uint32_t k0, k1;   // 0xFF where the code is >= 8: PRMT with selector bit 3 set replicates the selected byte's top bit
  asm("prmt.b32 %0, %1, %2, 0xD9C8;" : "=r"(k0) : "r"(q4), "r"(q));
  asm("prmt.b32 %0, %1, %2, 0xFBEA;" : "=r"(k1) : "r"(q4), "r"(q));
  asm("lop3.b32 %0, %1, %2, %3, 0xD8;" : "=r"(lo) : "r"(a0), "r"(b0), "r"(k0));     // k ? b : a
  asm("lop3.b32 %0, %1, %2, %3, 0xD8;" : "=r"(hi) : "r"(a1), "r"(b1), "r"(k1));
}
// four exponent bytes E and four raw bytes R (mantissa << 1 | sign) -> bf16 weights 0,1 in x and 2,3 in y
__device__ __forceinline__ void bf16x4(uint32_t R, uint32_t E, uint32_t &x, uint32_t &y) {
  const uint32_t p0 = __byte_perm(R, E, 0x5140), p1 = __byte_perm(R, E, 0x7362);     // [R0,E0,R1,E1], [R2,E2,R3,E3]
  asm("lop3.b32 %0, %1, %2, 0x7FFF7FFF, 0xE4;" : "=r"(x) : "r"(p0 >> 1), "r"(p0 << 15));
  asm("lop3.b32 %0, %1, %2, 0x7FFF7FFF, 0xE4;" : "=r"(y) : "r"(p1 >> 1), "r"(p1 << 15));
}
// Escape literals of one 4-step chunk: every escaped weight (code 15) takes the next word of the lane's own stream as its
// exponent byte, in weight order (the look-ahead word of the lane stream serves them like a renormalisation).
__device__ __forceinline__ void pair_literals(LaneStream &s, uint32_t esc /* bit 4n set: weight n escaped */, uint32_t dir,
                                              uint32_t &lo, uint32_t &hi) {
  while (esc) {
    const int n = (__ffs(int(esc)) - 1) >> 2;
    esc &= esc - 1;
    const uint32_t lit = s.w & 0xFFu;
    s.ptr += dir;
    asm volatile("ld.shared.u16 %0, [%1];" : "=r"(s.w) : "r"(s.ptr) : "memory");
    const uint32_t sh = 8u * uint32_t(n & 3), keep = ~(0xFFu << sh);
    if (n < 4) lo = (lo & keep) | (lit << sh);
    else hi = (hi & keep) | (lit << sh);
  }
}

// Raw-plane (bf16 sign+mantissa) reader of one tile: 16 steps of one lane = one 16-byte vector,
// fetched one vector ahead into registers, with an L2 prefetch four vectors ahead.
template <bool kPayload>
struct RawReader {
  const uint8_t *p;  // this lane's slice of the vector after `next`
  uint4 next;        // vector v + 1 while vector v is being consumed
  __device__ __forceinline__ uint4 load(int v, int V, int lane) {
    uint4 r;
    if (!kPayload || v < V - 1) {
      if (v + 4 < V) prefetch_l2(p + 4 * 512);
      r = ldg128_stream(p);
    } else {
      // last vector with the state-payload flag: 7 sub-rows of 32 x 2 bytes; bytes 14,15 come from the end state
      const uint16_t *q = reinterpret_cast<const uint16_t *>(p - 16 * lane) + lane;
      uint32_t h[7];
#pragma unroll
      for (int i = 0; i < 7; ++i) h[i] = q[i * 32];
      r.x = h[0] | (h[1] << 16); r.y = h[2] | (h[3] << 16); r.z = h[4] | (h[5] << 16); r.w = h[6];
    }
    p += 512;
    return r;
  }
  __device__ __forceinline__ void open(const uint8_t *tile_raw, int V, int lane) {
    p = tile_raw + 16 * lane;
    next = load(0, V, lane);
  }
  // returns vector v (already in `next`) and starts fetching v + 1
  __device__ __forceinline__ uint4 take(int v, int V, int lane) {
    const uint4 r = next;
    if (v + 1 < V) next = load(v + 1, V, lane);
    return r;
  }
};

// Decode one operand unit (32 operand bytes per row) of J tiles at once.
//   FMT: container format.  RB = tile_n / 32: the tile has RB row blocks of 32 rows and 2*RB chunk
//   rounds per unit; in round g lane l owns the 16-byte operand chunk (row (g % RB)*32 + l, half g / RB).
//   Emit: functor with
//     void chunk(int j, int g, int lane, uint4 v)    operand-format 16-byte chunk of stream j, round g, or
//     void packed(int j, int g, int lane, uint32_t b) for int4 when Emit::kOperand == false (4 packed bytes).
//   ring0: shared address of stream 0's ring (stream j's follows at j * kStreamSmem).
//   u: unit index inside the tile, V: raw vectors per tile (bf16).  sz[j]: int4: &(scale, zero)[group][first row of tile j].
//   POL: InterleavedWords (aux = lanemask_lt) or LaneWords (aux = this lane's cursor direction, +2 / -2).
template <uint32_t FMT, int RB, int J, bool kPayload, class POL, class Emit>
__device__ __forceinline__ void decode_unit(typename POL::S (&s)[J], uint32_t ring0, uint32_t tab, int lane, uint32_t lt, int u, int V,
                                            RawReader<kPayload> (&raw)[J], const uint32_t *const (&sz)[J], Emit &emit,
                                            const PairLut &pl = PairLut{0, 0, 0, 0}) {
  constexpr int G = 2 * RB;
  if constexpr (FMT == ANSLIN_FMT_BF16_PAIR4) {
    // one unit = 16 weights per row = 8 steps; a 4-step chunk = 8 weights = one 16-byte operand chunk; the chunk's escape
    // literals follow its last renormalisation.  32-row tiles and lane streams only (nothing else is ever launched).
    if constexpr (std::is_same<POL, LaneWords>::value && RB == 1) {
      uint4 rv[J];
#pragma unroll
      for (int j = 0; j < J; ++j) rv[j] = raw[j].take(u, V, lane);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        uint32_t q[J], esc[J], any = 0;
        decode4<POL, J>(s, q, tab, lt);
#pragma unroll
        for (int j = 0; j < J; ++j) {
          uint32_t t = q[j] & (q[j] >> 1);
          t &= t >> 2;
          esc[j] = t & 0x11111111u;   // nibble == 15
          any |= esc[j];
        }
        uint32_t lo[J], hi[J];
#pragma unroll
        for (int j = 0; j < J; ++j) pair_exps(q[j], pl, lo[j], hi[j]);
        if (__any_sync(0xffffffffu, any != 0)) {
#pragma unroll
          for (int j = 0; j < J; ++j) pair_literals(s[j], esc[j], lt, lo[j], hi[j]);
        }
#pragma unroll
        for (int j = 0; j < J; ++j) {
          uint4 o;
          bf16x4(h ? rv[j].z : rv[j].x, lo[j], o.x, o.y);
          bf16x4(h ? rv[j].w : rv[j].y, hi[j], o.z, o.w);
          if (kPayload && h == 1 && u == V - 1) {   // raw bytes 14, 15 of the last vector ride in the END state
            const uint32_t p2 = s[j].x - kL;
            o.w |= ((p2 >> 1) & 0x7Fu) | ((p2 & 1u) << 15) | (((p2 >> 9) & 0x7Fu) << 16) | (((p2 >> 8) & 1u) << 31);
          }
          emit.chunk(j, h, lane, o);
        }
      }
    }
  } else if constexpr (FMT == ANSLIN_FMT_BF16) {
#pragma unroll 1
    for (int g2 = 0; g2 < RB; ++g2) {  // two chunk rounds share one 16-byte raw vector
      const int v = u * RB + g2;
      uint4 rv[J];
#pragma unroll
      for (int j = 0; j < J; ++j) rv[j] = raw[j].take(v, V, lane);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        POL::template upkeep8<J>(s, ring0, lane);
        uint32_t R0[J], R1[J];
        uint4 o[J];
#pragma unroll
        for (int j = 0; j < J; ++j) { R0[j] = h ? rv[j].z : rv[j].x; R1[j] = h ? rv[j].w : rv[j].y; }
        if (kPayload && h == 1 && v == V - 1) {
          // last 8 steps of the tile: raw bytes 14,15 ride in the END state, known only after the last step, so
          // the last pair is decoded without raw bytes and they are merged in afterwards
          decode8_bf16<POL, J>(s, tab, lt, R0, R1, o);
#pragma unroll
          for (int j = 0; j < J; ++j) {
            const uint32_t pl = s[j].x - kL;   // byte 14 | byte 15 << 8, each = mantissa<<1 | sign
            o[j].w |= ((pl >> 1) & 0x7Fu) | ((pl & 1u) << 15) | (((pl >> 9) & 0x7Fu) << 16) | (((pl >> 8) & 1u) << 31);
          }
        } else {
          decode8_bf16<POL, J>(s, tab, lt, R0, R1, o);
        }
#pragma unroll
        for (int j = 0; j < J; ++j) emit.chunk(j, g2 * 2 + h, lane, o[j]);
      }
    }
  } else if constexpr (FMT == ANSLIN_FMT_INT4_AWQ) {
#pragma unroll 1
    for (int g = 0; g < G; ++g) {
      if ((g & 1) == 0) POL::template upkeep8<J>(s, ring0, lane);
      uint32_t B[J];
      decode4<POL, J>(s, B, tab, lt);
#pragma unroll
      for (int j = 0; j < J; ++j) {
        if constexpr (Emit::kOperand) {
          const uint32_t szv = __ldg(sz[j] + (g % RB) * 32 + lane);
          const __half2 szh = *reinterpret_cast<const __half2 *>(&szv);
          const __half2 sc = __half2half2(__low2half(szh));
          const __half2 zoff = __hadd2(__half2half2(__high2half(szh)), __float2half2_rn(1024.f));
          emit.chunk(j, g, lane, make_uint4(awq_dequant2(B[j] & 0xFF, zoff, sc), awq_dequant2((B[j] >> 8) & 0xFF, zoff, sc),
                                            awq_dequant2((B[j] >> 16) & 0xFF, zoff, sc), awq_dequant2(B[j] >> 24, zoff, sc)));
        } else {
          emit.packed(j, g, lane, B[j]);
        }
      }
    }
  } else if constexpr (FMT == ANSLIN_FMT_FP4_E2M1) {
#pragma unroll 1
    for (int g = 0; g < G; ++g) {   // 8 packed bytes = 16 codes = one 16-byte chunk of e4m3 operand bytes
      POL::template upkeep8<J>(s, ring0, lane);
      uint32_t B0[J], B1[J];
      decode4<POL, J>(s, B0, tab, lt);
      decode4<POL, J>(s, B1, tab, lt);
#pragma unroll
      for (int j = 0; j < J; ++j) {
        if constexpr (Emit::kOperand) {
          uint4 v;
          e2m1x8_to_e4m3(B0[j], v.x, v.y);
          e2m1x8_to_e4m3(B1[j], v.z, v.w);
          emit.chunk(j, g, lane, v);
        } else {
          emit.packed8(j, g, lane, B0[j], B1[j]);
        }
      }
    }
  } else {  // fp8 / int8: the byte is the operand
#pragma unroll 1
    for (int g = 0; g < G; ++g) {
      uint32_t q0[J], q1[J], q2[J], q3[J];
      POL::template upkeep8<J>(s, ring0, lane);
      decode4<POL, J>(s, q0, tab, lt);
      decode4<POL, J>(s, q1, tab, lt);
      POL::template upkeep8<J>(s, ring0, lane);
      decode4<POL, J>(s, q2, tab, lt);
      decode4<POL, J>(s, q3, tab, lt);
#pragma unroll
      for (int j = 0; j < J; ++j) emit.chunk(j, g, lane, make_uint4(q0[j], q1[j], q2[j], q3[j]));
    }
  }
}

}  // namespace anslin
