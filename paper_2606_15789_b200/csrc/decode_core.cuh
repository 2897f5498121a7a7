// Warp-cooperative rANS tile decoder (Alg V.2, P:l.260-287), sm_100a.
//
// One warp decodes one tile: lane l owns stream l (P:l.192 "each warp lane maintains its own rANS
// state").  Per step and lane:  slot = x & 4095;  e = T[slot] (shared-memory table, P:l.271);
// x = f*(x>>12) + bias;  if x < 2^16: x = x<<16 | next word.  The words of a tile are interleaved
// in decoder read order, so the renormalising lanes of a step read CONSECUTIVE 16-bit words
// (P:l.256 "renormalization loads are naturally coalesced"): ballot + popc prefix picks the word.
// The compressed words are streamed HBM -> shared memory through a per-warp 2 KiB ring with
// 16-byte cp.async (32 lanes x 16 B = 512 B per fill, 1.5-2 KiB of look-ahead); the ring
// bookkeeping runs once per EIGHT decode steps.
//
// Table entry (4 B, Eq.3's "2^b x 4 B", P:l.440):  sym[7:0] | f[19:8] | bias[31:20].
#pragma once
#include <cuda_fp16.h>
#include <stdint.h>
#include "anslin_internal.h"

namespace anslin {

constexpr uint32_t kRingBytes = 2048;  // per decoder warp; the ring must be 2 KiB aligned
constexpr uint32_t kFillBytes = 512;   // 32 lanes x 16 B per fill
// The ring reads ahead of the record it decodes: the container guarantees this many readable bytes
// after the records section (tail rule), so fills need no bounds check.
static_assert(2 * kRingBytes <= uint32_t(kTailBytes), "ring read-ahead must fit the container tail rule");

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}
__device__ __forceinline__ uint32_t lds16(uint32_t a) {
  uint16_t v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t a, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
// 16-byte cp.async, executed only when `on` != 0; copies src_bytes (16 or 0 = zero fill) bytes.
__device__ __forceinline__ void cp_async16_if(uint32_t on, uint32_t dst, const void *src, uint32_t src_bytes) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0;\n\t@p cp.async.cg.shared.global [%1], [%2], 16, %3;\n\t}" ::"r"(on), "r"(dst),
      "l"(src), "r"(src_bytes)
      : "memory");
}
__device__ __forceinline__ void cp_async_commit_if(uint32_t on) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %0, 0;\n\t@p cp.async.commit_group;\n\t}" ::"r"(on) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }
__device__ __forceinline__ uint32_t lds32(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ uint4 ldg128_stream(const void *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// Expand the 256 x u16 frequency table of the container into the 4096-entry slot table in shared
// memory (Alg V.1 l.6 "Copy global decode table T into shared memory", P:l.212).  All threads of
// the CTA must call; `cum` is 257 u32 of scratch.  Ends with __syncthreads().
__device__ __forceinline__ void build_slot_table(uint32_t *tab, uint32_t *cum, const uint16_t *freq_g) {
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
  if (warp == 0) {  // exclusive prefix sum of 256 frequencies: 8 per lane + warp scan
    uint32_t f[8], s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { f[i] = freq_g[lane * 8 + i]; s += f[i]; }
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
    for (uint32_t k = lane; k < f; k += 32) tab[c0 + k] = uint32_t(s) | (f << 8) | (k << 20);
  }
  __syncthreads();
}

// Per-warp stream state over one tile record.
struct WarpStream {
  uint32_t x;       // this lane's rANS state
  uint32_t posb;    // BYTES of words consumed so far (warp uniform)
  uint32_t filled;  // bytes of words whose ring fill has been issued (warp uniform, multiple of 512)
  uint32_t ring;    // shared-space address of this warp's 2 KiB-aligned ring
  const uint8_t *src;  // this lane's next fill source = words + filled + 16*lane
};

// Issue the next 512-byte ring fill iff `on` (every lane copies 16 B).
__device__ __forceinline__ void stream_fill_if(WarpStream &s, uint32_t on, int lane) {
  cp_async16_if(on, s.ring | ((s.filled + (uint32_t(lane) << 4)) & (kRingBytes - 1)), s.src, 16u);
  cp_async_commit_if(on);
  s.filled += on ? kFillBytes : 0u;
  s.src += on ? kFillBytes : 0u;
}

// rec = start of the tile record in HBM (16-byte aligned).
__device__ __forceinline__ void stream_open(WarpStream &s, const uint8_t *rec, uint32_t ring, int lane) {
  cp_async_wait_all();  // fills of the previous tile may still be in flight into this ring
  __syncwarp();
  s.x = reinterpret_cast<const uint32_t *>(rec)[lane];
  s.src = rec + 4 * kLanes + 16 * lane;
  s.posb = 0; s.filled = 0; s.ring = ring;
#pragma unroll
  for (int i = 0; i < 4; ++i) stream_fill_if(s, 1u, lane);
}

// Ring upkeep for the next EIGHT decode steps (they consume at most 512 B): refill the dead quarter
// behind the read position and make sure everything up to posb + 1024 has landed.  Invariant:
// 1536 <= filled - posb <= 2048 after the call, at most ONE fill pending => landed >= posb + 1024
// >= the 512 + 62 bytes eight steps can touch.  A fill writes ring bytes
// [filled, filled + 512) - 2048 < posb, i.e. only words already consumed.
__device__ __forceinline__ void stream_upkeep8(WarpStream &s, int lane) {
  stream_fill_if(s, uint32_t(s.filled - s.posb < 1536u), lane);
  cp_async_wait_1();
  __syncwarp();
}

// One decode step of Alg V.2 for all 32 lanes; returns the table entry (symbol in bits 7:0).
__device__ __forceinline__ uint32_t decode_step(WarpStream &s, uint32_t tab_s, uint32_t lt) {
  uint32_t ea;
  asm("mad.lo.u32 %0, %1, 4, %2;" : "=r"(ea) : "r"(s.x & (kM - 1)), "r"(tab_s));
  const uint32_t e = lds32(ea);
  const uint32_t xn = ((e >> 8) & 0xFFFu) * (s.x >> kProbBits) + (e >> 20);
  const bool need = xn < kL;
  const uint32_t mask = __ballot_sync(0xffffffffu, need);
  // every lane loads (the window is resident); only renormalising lanes use the word
  const uint32_t w = lds16(s.ring | ((s.posb + 2u * __popc(mask & lt)) & (kRingBytes - 1)));
  s.x = need ? __byte_perm(w, xn, 0x5410) : xn;  // (xn << 16) | w
  s.posb += 2u * __popc(mask);
  return e;
}

// Insert the symbol byte of table entry e at byte position `pos` of acc.
template <int pos>
__device__ __forceinline__ uint32_t put_sym(uint32_t acc, uint32_t e) {
  return __byte_perm(acc, e, (0x3210 & ~(0xF << (4 * pos))) | (4 << (4 * pos)));
}
// Four decode steps -> four symbol bytes.
__device__ __forceinline__ uint32_t decode4(WarpStream &s, uint32_t tab, uint32_t lt) {
  uint32_t q = 0;
  q = put_sym<0>(q, decode_step(s, tab, lt));
  q = put_sym<1>(q, decode_step(s, tab, lt));
  q = put_sym<2>(q, decode_step(s, tab, lt));
  q = put_sym<3>(q, decode_step(s, tab, lt));
  return q;
}

// bf16: merge 4 exponent bytes (E) with 4 raw bytes (R = mantissa<<1 | sign) into 4 bf16 values.
__device__ __forceinline__ uint2 bf16_merge4(uint32_t E, uint32_t R) {
  const uint32_t p0 = __byte_perm(R, E, 0x5140), p1 = __byte_perm(R, E, 0x7362);
  uint2 o;
  o.x = ((p0 >> 1) & 0x7FFF7FFFu) | ((p0 << 15) & 0x80008000u);
  o.y = ((p1 >> 1) & 0x7FFF7FFFu) | ((p1 << 15) & 0x80008000u);
  return o;
}

// int4 (AWQ-style): one packed byte (low nibble = even k) -> two fp16 weights (q - z) * s.
// 0x6400 | q is the fp16 number 1024 + q, so (1024+q) - (1024+z) is exact and the product rounds once.
__device__ __forceinline__ uint32_t awq_dequant2(uint32_t byte, __half2 zoff, __half2 sc) {
  const uint32_t v = (byte & 0x0Fu) | ((byte & 0xF0u) << 12) | 0x64006400u;
  __half2 h = *reinterpret_cast<const __half2 *>(&v);
  h = __hmul2(__hsub2(h, zoff), sc);
  return *reinterpret_cast<const uint32_t *>(&h);
}

// Raw-plane (bf16 sign+mantissa) reader: 16 steps of one lane = one 16-byte vector.
template <bool kPayload>
struct RawReader {
  const uint8_t *tile_raw;
  int V;  // vectors per tile
  __device__ __forceinline__ uint4 load(int v, int lane) const {
    if (!kPayload || v < V - 1) return ldg128_stream(tile_raw + size_t(v) * 512 + lane * 16);
    // last vector with the state-payload flag: 7 sub-rows of 32 x 2 bytes; bytes 14,15 come from the end state
    uint32_t h[7];
#pragma unroll
    for (int i = 0; i < 7; ++i)
      h[i] = reinterpret_cast<const uint16_t *>(tile_raw + size_t(v) * 512)[i * 32 + lane];
    uint4 r;
    r.x = h[0] | (h[1] << 16); r.y = h[2] | (h[3] << 16); r.z = h[4] | (h[5] << 16); r.w = h[6];
    return r;
  }
};

// Decode one operand unit (128 rows x 32 operand bytes = 256 chunks of 16 B) of a tile.
//   FMT: container format.  Emit: functor with
//     void chunk(int g, int lane, uint4 v)   operand-format 16-byte chunk of round g (all formats), or
//     void packed(int g, int lane, uint32_t b) for int4 when Emit::kOperand == false (4 packed bytes).
//   u: unit index inside the tile (selects the raw vectors / scale group).
template <uint32_t FMT, bool kPayload, class Emit>
__device__ __forceinline__ void decode_unit(WarpStream &s, uint32_t tab, int lane, uint32_t lt, int u,
                                            const RawReader<kPayload> &raw, uint4 &raw_next, uint4 &raw_next2,
                                            const uint32_t *sz_row /* int4: &sz[group][n0] */, Emit &emit) {
  if constexpr (FMT == ANSLIN_FMT_BF16) {
#pragma unroll 1
    for (int g2 = 0; g2 < 4; ++g2) {  // two rounds share one 16-byte raw vector; vectors are fetched two ahead
      const int v = u * 4 + g2;
      uint4 rv = raw_next;
      raw_next = raw_next2;
      if (v + 2 < raw.V) raw_next2 = raw.load(v + 2, lane);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        stream_upkeep8(s, lane);
        const uint32_t E0 = decode4(s, tab, lt), E1 = decode4(s, tab, lt);
        if (kPayload && v == raw.V - 1 && h == 1) {  // last 8 steps of the tile: bytes 14,15 ride in the state
          const uint32_t p = s.x - kL;
          rv.w = (rv.w & 0xFFFFu) | (p << 16);
        }
        const uint2 a = bf16_merge4(E0, h ? rv.z : rv.x), b = bf16_merge4(E1, h ? rv.w : rv.y);
        emit.chunk(g2 * 2 + h, lane, make_uint4(a.x, a.y, b.x, b.y));
      }
    }
  } else if constexpr (FMT == ANSLIN_FMT_INT4_AWQ) {
#pragma unroll 1
    for (int g = 0; g < 8; ++g) {
      if ((g & 1) == 0) stream_upkeep8(s, lane);
      const uint32_t B = decode4(s, tab, lt);
      if constexpr (Emit::kOperand) {
        const uint32_t szv = __ldg(sz_row + (g & 3) * 32 + lane);
        const __half2 sz = *reinterpret_cast<const __half2 *>(&szv);
        const __half2 sc = __half2half2(__low2half(sz));
        const __half2 zoff = __hadd2(__half2half2(__high2half(sz)), __float2half2_rn(1024.f));
        emit.chunk(g, lane, make_uint4(awq_dequant2(B & 0xFF, zoff, sc), awq_dequant2((B >> 8) & 0xFF, zoff, sc),
                                       awq_dequant2((B >> 16) & 0xFF, zoff, sc), awq_dequant2(B >> 24, zoff, sc)));
      } else {
        emit.packed(g, lane, B);
      }
    }
  } else {  // fp8 / int8: the byte is the operand
#pragma unroll 1
    for (int g = 0; g < 8; ++g) {
      stream_upkeep8(s, lane);
      const uint32_t q0 = decode4(s, tab, lt), q1 = decode4(s, tab, lt);
      stream_upkeep8(s, lane);
      const uint32_t q2 = decode4(s, tab, lt), q3 = decode4(s, tab, lt);
      emit.chunk(g, lane, make_uint4(q0, q1, q2, q3));
    }
  }
}

}  // namespace anslin
