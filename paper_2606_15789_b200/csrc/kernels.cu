// libanslin device side (sm_100a): decode-only kernel, fused rANS-decode + tcgen05 GEMM kernel,
// dense tcgen05 comparator, and their C-ABI launchers.
//
// Fused kernel = Alg V.1 (P:l.196-252) re-designed for Blackwell (DESIGN.md §"Kernels"):
//   * the paper's single producer warp becomes up to 24 decoder warps per CTA (decode is the
//     bottleneck at small batch, P:l.306), each running Alg V.2 on its own tile;
//   * the paper's consumer warps become ONE thread issuing tcgen05.mma with the accumulator in
//     TMEM; the weights are the MMA "A" operand (M = 128 weight rows), the batch is MMA N;
//   * ready[2] flags (P:l.210) become mbarrier full/empty pairs over a ring of 4 KiB operand
//     units (128 rows x 32 B = one MMA K step), so a decoder warp hands the tensor core a K slice
//     every 64 (bf16) decode steps instead of a whole tile ("ring buffer lets decode run several
//     sub-tiles ahead", P:l.297);
//   * activations arrive by TMA (cp.async.bulk.tensor) into the same ring slot.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "anslin_internal.h"
#include "decode_core.cuh"

using namespace anslin;

namespace {

thread_local int g_launches = 0;

// ------------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// Bounded wait: a protocol bug traps (launch failure) instead of hanging the GPU.
// kSleepNs > 0 backs off between probes so that long waits (MMA issuer, epilogue) do not steal issue
// slots from the decoder warps sharing their scheduler.
template <int kSleepNs = 0>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0, spins = 0;
  while (true) {
    if (kSleepNs > 0 && spins > 0) __nanosleep(kSleepNs);
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    if (done) break;
    if (++spins > (1u << 26)) __trap();
  }
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
template <int KIND>  // 0 = f16 (bf16/fp16), 1 = f8f6f4, 2 = i8
__device__ __forceinline__ void umma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  if constexpr (KIND == 0)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
                 "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
                 : "memory");
  else if constexpr (KIND == 1)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
                 "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
                 : "memory");
  else
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
                 "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
                 : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// UMMA shared-memory descriptor, K-major (cute::UMMA::SmemDescriptor bit layout):
// start>>4 [0,14) | LBO>>4 [16,30) | SBO>>4 [32,46) | version=1 [46,48) | layout [61,64)
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout) {
  return uint64_t((addr >> 4) & 0x3FFF) | (uint64_t((lbo_bytes >> 4) & 0x3FFF) << 16) |
         (uint64_t((sbo_bytes >> 4) & 0x3FFF) << 32) | (uint64_t(1) << 46) | (uint64_t(layout) << 61);
}
constexpr uint32_t kLayoutNone = 0, kLayoutSW128 = 2, kLayoutSW32 = 6;

// Instruction descriptor (cute::UMMA::InstrDescriptor): c_format [4,6) a_format [7,10) b_format [10,13)
// a/b major = K (0) | N>>3 [17,23) | M>>4 [24,29)
__host__ __device__ constexpr uint32_t make_idesc(uint32_t cfmt, uint32_t afmt, uint32_t bfmt, uint32_t M, uint32_t N) {
  return (cfmt << 4) | (afmt << 7) | (bfmt << 10) | ((N >> 3) << 17) | ((M >> 4) << 24);
}
template <uint32_t FMT> struct FmtTraits;
template <> struct FmtTraits<ANSLIN_FMT_BF16> { static constexpr int kind = 0; static constexpr uint32_t c = 1, ab = 1; static constexpr int xbytes = 2; };
template <> struct FmtTraits<ANSLIN_FMT_INT4_AWQ> { static constexpr int kind = 0; static constexpr uint32_t c = 1, ab = 0; static constexpr int xbytes = 2; };
template <> struct FmtTraits<ANSLIN_FMT_FP8_E4M3> { static constexpr int kind = 1; static constexpr uint32_t c = 1, ab = 0; static constexpr int xbytes = 1; };
template <> struct FmtTraits<ANSLIN_FMT_INT8> { static constexpr int kind = 2; static constexpr uint32_t c = 2, ab = 1; static constexpr int xbytes = 1; };

// ------------------------------------------------------------------------------------------------
// Parameters
// ------------------------------------------------------------------------------------------------
struct ContainerView {
  const uint8_t *base;
  uint64_t off_freq, off_offsets, off_records, off_raw, off_scales, total;
  uint32_t n_out, k_in, tile_k, KT, n_tiles, units, group, flags;
  float w_scale;
};

ContainerView view_of(const anslin_weight *w) {
  const Header &h = w->h;
  ContainerView v;
  v.base = w->dev;
  v.off_freq = h.off_freq; v.off_offsets = h.off_offsets; v.off_records = h.off_records; v.off_raw = h.off_raw;
  v.off_scales = h.off_scales; v.total = h.total_bytes;
  v.n_out = h.n_out; v.k_in = h.k_in; v.tile_k = h.tile_k; v.KT = h.k_in / h.tile_k; v.n_tiles = h.n_tiles;
  v.units = h.tile_k / unit_k_of(h.format); v.group = h.group_size; v.flags = h.flags; v.w_scale = h.w_scale;
  return v;
}

// ------------------------------------------------------------------------------------------------
// Decode-only kernel (anslin_decode): one warp per tile, output row-major W to HBM.
// ------------------------------------------------------------------------------------------------
template <uint32_t FMT>
struct GlobalEmit {
  static constexpr bool kOperand = false;
  uint8_t *tile_out;  // &W[n0][k0] in bytes
  size_t row_bytes;   // bytes per W row
  int u;
  __device__ __forceinline__ void chunk(int g, int lane, uint4 v) const {  // bf16 / fp8 / int8: 16 B of row-major W
    uint8_t *p = tile_out + size_t((g & 3) * 32 + lane) * row_bytes + size_t(u) * 32 + (g >> 2) * 16;
    *reinterpret_cast<uint4 *>(p) = v;
  }
  __device__ __forceinline__ void packed(int g, int lane, uint32_t b) const {  // int4: 4 packed bytes = 8 weights
    uint8_t *p = tile_out + size_t((g & 3) * 32 + lane) * row_bytes + size_t(u) * 8 + (g >> 2) * 4;
    *reinterpret_cast<uint32_t *>(p) = b;
  }
};

constexpr int kDecWarps = 8;

template <uint32_t FMT, bool PAYLOAD>
__global__ void __launch_bounds__(kDecWarps * 32) decode_kernel(ContainerView cv, uint8_t *out) {
  __shared__ __align__(16) uint32_t tab[kM];
  __shared__ uint32_t cum[260];
  __shared__ __align__(16) uint8_t rings[(kDecWarps + 1) * kRingBytes];  // +1: rounded up to ring-size alignment below
  build_slot_table(tab, cum, reinterpret_cast<const uint16_t *>(cv.base + cv.off_freq));
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t lt = lanemask_lt(), ring_s = ((smem_u32(rings) + kRingBytes - 1) & ~(kRingBytes - 1)) + uint32_t(warp) * kRingBytes;
  const uint32_t *offs = reinterpret_cast<const uint32_t *>(cv.base + cv.off_offsets);
  const size_t row_bytes = FMT == ANSLIN_FMT_BF16 ? size_t(cv.k_in) * 2 : FMT == ANSLIN_FMT_INT4_AWQ ? size_t(cv.k_in) / 2 : size_t(cv.k_in);
  const size_t tile_row_bytes = FMT == ANSLIN_FMT_BF16 ? size_t(cv.tile_k) * 2 : FMT == ANSLIN_FMT_INT4_AWQ ? size_t(cv.tile_k) / 2 : size_t(cv.tile_k);
  const size_t rtb = raw_tile_bytes(kTileN, cv.tile_k, PAYLOAD ? ANSLIN_FLAG_STATE_PAYLOAD : 0);
  for (uint32_t t = blockIdx.x * kDecWarps + warp; t < cv.n_tiles; t += gridDim.x * kDecWarps) {
    WarpStream s;
    stream_open(s, cv.base + cv.off_records + size_t(offs[t]) * 16, ring_s, lane);
    const uint32_t stripe = t / cv.KT, kt = t % cv.KT;
    GlobalEmit<FMT> emit;
    emit.tile_out = out + size_t(stripe) * kTileN * row_bytes + size_t(kt) * tile_row_bytes;
    emit.row_bytes = row_bytes;
    RawReader<PAYLOAD> raw;
    raw.tile_raw = cv.base + cv.off_raw + size_t(t) * rtb;
    raw.V = int(cv.units) * 4;
    uint4 raw_next = make_uint4(0, 0, 0, 0), raw_next2 = raw_next;
    if (FMT == ANSLIN_FMT_BF16) { raw_next = raw.load(0, lane); raw_next2 = raw.load(1, lane); }
    for (uint32_t u = 0; u < cv.units; ++u) {
      emit.u = int(u);
      decode_unit<FMT, PAYLOAD>(s, smem_u32(tab), lane, lt, int(u), raw, raw_next, raw_next2, nullptr, emit);
    }
  }
  cp_async_wait_all();
}

// ------------------------------------------------------------------------------------------------
// Fused decode + GEMM kernel
// ------------------------------------------------------------------------------------------------
constexpr int kEpiWarps = 4;
constexpr int kMmaWarp = 4;
constexpr int kFirstDecWarp = 5;
constexpr int kMaxDecWarps = 24;
constexpr int kGemmThreads = 32 * (kFirstDecWarp + kMaxDecWarps);
constexpr int kMaxSlots = 48;

struct GemmParams {
  ContainerView cv;
  const float *x_scale;    // int8 / fp8: f32[m]
  float *y;
  int64_t ldy;
  uint32_t *partials;      // [2*grid][mpad][128] raw accumulator bits
  uint32_t *counters;      // [stripes]
  uint32_t m, mpad;
  uint32_t U, D;           // ring slots, decoder warps
  uint32_t slot_bytes;     // 4096 + mpad*32
  uint32_t tmem_cols;
  uint32_t layout;         // kLayoutSW32 or kLayoutNone (debug alternative)
};

// Shared-memory unit slot writer: the decoded 16-byte chunk goes where the UMMA K-major canonical
// layout expects it (P:l.151 "consumed by the GEMM kernel in its required swizzled layout").
struct SmemEmit {
  static constexpr bool kOperand = true;
  uint32_t slot_a;   // shared address of the unit's A operand (4 KiB)
  uint32_t layout;
  __device__ __forceinline__ void chunk(int g, int lane, uint4 v) const {
    const uint32_t row = uint32_t((g & 3) * 32 + lane), c = uint32_t(g >> 2);
    uint32_t a;
    if (layout == kLayoutSW32) a = slot_a + row * 32u + ((c ^ ((uint32_t(lane) >> 2) & 1u)) << 4);  // Swizzle<1,4,3>
    else a = slot_a + c * 2048u + row * 16u;                                                        // 8x16B core matrices
    sts128(a, v);
  }
  __device__ __forceinline__ void packed(int, int, uint32_t) const {}
};

struct Segment { uint32_t stripe, ka, nt; };

// Work of CTA c: tiles [t0, t1) of the stripe-major tile sequence (stream-K style equal split).
__device__ __forceinline__ uint32_t cta_first_tile(uint32_t c, uint32_t G, uint32_t T) { return uint32_t(uint64_t(c) * T / G); }
__device__ __forceinline__ uint32_t cta_of_tile(uint32_t t, uint32_t G, uint32_t T) {  // largest c with first_tile(c) <= t
  return uint32_t((uint64_t(t + 1) * G + T - 1) / T) - 1;
}

template <uint32_t FMT>
__device__ __forceinline__ float finalize(uint32_t bits, float xs, float ws) {
  if constexpr (FMT == ANSLIN_FMT_INT8) return float(int32_t(bits)) * xs * ws;
  else if constexpr (FMT == ANSLIN_FMT_FP8_E4M3) return __uint_as_float(bits) * xs * ws;
  else return __uint_as_float(bits);
}
template <uint32_t FMT>
__device__ __forceinline__ uint32_t acc_add(uint32_t a, uint32_t b) {
  if constexpr (FMT == ANSLIN_FMT_INT8) return uint32_t(int32_t(a) + int32_t(b));
  else return __float_as_uint(__uint_as_float(a) + __uint_as_float(b));
}


// ------------------------------------------------------------------------------------------------
// Epilogue (a10), shared by the fused and the dense kernel.  Warps 0..3: TMEM -> registers -> Y for
// whole stripes, or -> split-K partial + deterministic fix-up (the LAST CTA to finish a stripe sums
// all partials in CTA order, 16-byte loads, up to 8 contributors in flight per thread).
// ------------------------------------------------------------------------------------------------
struct EpiParams {
  const float *x_scale;     // int8 / fp8: f32[m]
  const __half *w_scale_h;  // int8: fp16[n_out]
  float w_scale;            // fp8
  float *y;
  int64_t ldy;
  uint32_t *partials, *counters;
  uint32_t m, mpad;
};

__device__ __forceinline__ uint4 ldcg128(const uint32_t *p) {
  uint4 r;
  asm volatile("ld.global.cg.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

template <uint32_t FMT>
__device__ __forceinline__ void epilogue_run(const EpiParams &p, uint32_t tmem_base, uint32_t tfull_s, uint32_t tempty_s,
                                             volatile uint32_t *flag, uint32_t t_begin, uint32_t t_end, uint32_t KT, uint32_t G,
                                             uint32_t T, int warp, int lane) {
  constexpr bool kScaled = FMT == ANSLIN_FMT_INT8 || FMT == ANSLIN_FMT_FP8_E4M3;
  const uint32_t row = uint32_t(warp * 32 + lane);
  uint32_t si = 0;
  for (uint32_t t = t_begin; t < t_end; ++si) {
    const uint32_t stripe = t / KT, ka = t % KT, nt = min(KT - ka, t_end - t), ab = si & 1u;
    const bool whole = (ka == 0 && nt == KT);
    const uint32_t n = stripe * kTileN + row;
    float ws = 1.0f;
    if (FMT == ANSLIN_FMT_INT8) ws = __half2float(p.w_scale_h[n]);
    if (FMT == ANSLIN_FMT_FP8_E4M3) ws = p.w_scale;
    mbar_wait<400>(tfull_s + 8 * ab, (si >> 1) & 1u);
    tc_fence_after();
    const uint32_t pslot = blockIdx.x * 2u + (t == t_begin ? 0u : 1u);
    uint32_t *part = p.partials + size_t(pslot) * p.mpad * kTileN;
    for (uint32_t c0 = 0; c0 < p.mpad; c0 += 16) {
      uint32_t v[16];
      tmem_ld16(tmem_base + ((uint32_t(warp) * 32u) << 16) + ab * p.mpad + c0, v);
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const uint32_t mm = c0 + j;
        if (mm < p.m) {
          if (whole) p.y[size_t(mm) * p.ldy + n] = finalize<FMT>(v[j], kScaled ? p.x_scale[mm] : 1.0f, ws);
          else part[size_t(mm) * kTileN + row] = v[j];
        }
      }
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(tempty_s + 8 * ab);
    if (!whole) {
      const uint32_t c_first = cta_of_tile(stripe * KT, G, T), c_last = cta_of_tile(stripe * KT + KT - 1, G, T);
      __threadfence();
      named_bar_sync(1, kEpiWarps * 32);
      if (threadIdx.x == 0) *flag = (atomicAdd(&p.counters[stripe], 1u) == c_last - c_first) ? 1u : 0u;
      named_bar_sync(1, kEpiWarps * 32);
      if (*flag) {
        __threadfence();
        // thread -> 4 consecutive output channels (one 16-byte load per contributor), warp -> batch rows mm = warp, warp+4, ..
        const uint32_t r4 = uint32_t(lane) * 4u, n4 = stripe * kTileN + r4;
        float ws4[4] = {ws, ws, ws, ws};
        if (FMT == ANSLIN_FMT_INT8)
#pragma unroll
          for (int j = 0; j < 4; ++j) ws4[j] = __half2float(p.w_scale_h[n4 + j]);
        for (uint32_t mm = uint32_t(warp); mm < p.m; mm += kEpiWarps) {
          uint32_t acc[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) acc[j] = FMT == ANSLIN_FMT_INT8 ? 0u : __float_as_uint(0.0f);
          for (uint32_t cb = c_first; cb <= c_last; cb += 8) {
            uint4 v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const uint32_t c = cb + j;
              v[j] = make_uint4(0, 0, 0, 0);
              if (c <= c_last) {
                const uint32_t ps = c * 2u + (cta_first_tile(c, G, T) / KT == stripe ? 0u : 1u);
                v[j] = ldcg128(p.partials + (size_t(ps) * p.mpad + mm) * kTileN + r4);
              }
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) {  // fixed CTA order -> bit-reproducible sums
              acc[0] = acc_add<FMT>(acc[0], v[j].x); acc[1] = acc_add<FMT>(acc[1], v[j].y);
              acc[2] = acc_add<FMT>(acc[2], v[j].z); acc[3] = acc_add<FMT>(acc[3], v[j].w);
            }
          }
          const float xs = kScaled ? p.x_scale[mm] : 1.0f;
          float *yo = p.y + size_t(mm) * p.ldy + n4;
#pragma unroll
          for (int j = 0; j < 4; ++j) yo[j] = finalize<FMT>(acc[j], xs, ws4[j]);
        }
        if (threadIdx.x == 0) p.counters[stripe] = 0;
      }
      named_bar_sync(1, kEpiWarps * 32);  // flag is reused by the next segment
    }
    t += nt;
  }
}

template <uint32_t FMT, bool PAYLOAD>
__global__ void __launch_bounds__(kGemmThreads, 1) fused_gemm_kernel(const __grid_constant__ CUtensorMap tmx, GemmParams p) {
  using TR = FmtTraits<FMT>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 2047u) & ~2047u;
  uint8_t *smem = smem_raw + (smem0 - smem_u32(smem_raw));
  // carve-up
  const uint32_t slots_s = smem0;
  const uint32_t ring_off = (p.U * p.slot_bytes + kRingBytes - 1) & ~(kRingBytes - 1);   // rings are ring-size aligned
  const uint32_t tab_off = ring_off + p.D * kRingBytes;
  uint32_t *tab = reinterpret_cast<uint32_t *>(smem + tab_off);
  uint32_t *cum = reinterpret_cast<uint32_t *>(smem + tab_off + 16384);
  const uint32_t bar_off = tab_off + 16384 + 1056;
  const uint32_t full_s = smem0 + bar_off, empty_s = full_s + 8 * kMaxSlots, tfull_s = empty_s + 8 * kMaxSlots,
                 tempty_s = tfull_s + 16, tmemptr_s = tempty_s + 16, flag_s = tmemptr_s + 8;
  volatile uint32_t *tmemptr = reinterpret_cast<volatile uint32_t *>(smem + bar_off + 16 * kMaxSlots + 32);
  volatile uint32_t *flag = reinterpret_cast<volatile uint32_t *>(smem + bar_off + 16 * kMaxSlots + 40);
  // lapw[slot] = number of ring laps whose producer has ACQUIRED the slot.  A decoder warp may run
  // more than one lap ahead of a slot's barrier (idle rounds, segment changes), where an mbarrier
  // parity wait would alias; it first waits for its predecessor lap to be acquired.
  volatile uint32_t *lapw = reinterpret_cast<volatile uint32_t *>(smem + bar_off + 16 * kMaxSlots + 64);

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const ContainerView &cv = p.cv;
  const uint32_t G = gridDim.x, T = cv.n_tiles, KT = cv.KT;

  if (threadIdx.x == 0) {
    for (uint32_t i = 0; i < p.U; ++i) { mbar_init(full_s + 8 * i, 2); mbar_init(empty_s + 8 * i, 1); lapw[i] = 0; }
    for (uint32_t i = 0; i < 2; ++i) { mbar_init(tfull_s + 8 * i, 1); mbar_init(tempty_s + 8 * i, kEpiWarps); }
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc(tmemptr_s, p.tmem_cols);
  tc_fence_before();
  build_slot_table(tab, cum, reinterpret_cast<const uint16_t *>(cv.base + cv.off_freq));  // ends with __syncthreads()
  tc_fence_after();
  const uint32_t tmem_base = *tmemptr;

  const uint32_t t_begin = cta_first_tile(blockIdx.x, G, T), t_end = cta_first_tile(blockIdx.x + 1, G, T);
  const uint32_t units = cv.units;

  if (warp >= kFirstDecWarp) {
    // ===================== decoder warps: Alg V.2 into the operand ring =====================
    const uint32_t d = uint32_t(warp - kFirstDecWarp);
    if (d < p.D) {
      const uint32_t lt = lanemask_lt(), ring_s = smem0 + ring_off + d * kRingBytes;
      const uint32_t *offs = reinterpret_cast<const uint32_t *>(cv.base + cv.off_offsets);
      const size_t rtb = raw_tile_bytes(kTileN, cv.tile_k, PAYLOAD ? ANSLIN_FLAG_STATE_PAYLOAD : 0);
      const uint32_t xbytes = p.mpad * 32u;
      // Tiles of this CTA are dealt to the decoder warps round-robin over the CTA's WHOLE range
      // (tile i -> warp i mod D, round i div D).  The MMA warp consumes units segment by segment
      // (one accumulator per stripe segment); inside a segment the order is (round, unit, tile).
      for (uint32_t i = d; i < t_end - t_begin; i += p.D) {
        const uint32_t gt = t_begin + i, stripe = gt / KT, kt = gt % KT;
        const uint32_t seg_a = max(t_begin, stripe * KT) - t_begin;            // segment = [seg_a, seg_b) in CTA-local tiles
        const uint32_t seg_b = min(t_end, stripe * KT + KT) - t_begin;
        const uint32_t rho = i / p.D;
        const uint32_t grp_a = max(seg_a, rho * p.D), grp_b = min(seg_b, rho * p.D + p.D);   // this round's tiles of the segment
        const uint32_t seq0 = (seg_a + (grp_a - seg_a)) * units, cnt = grp_b - grp_a, idx = i - grp_a;
        WarpStream s;
        stream_open(s, cv.base + cv.off_records + size_t(offs[gt]) * 16, ring_s, lane);
        RawReader<PAYLOAD> raw;
        raw.tile_raw = cv.base + cv.off_raw + size_t(gt) * rtb;
        raw.V = int(units) * 4;
        uint4 raw_next = make_uint4(0, 0, 0, 0), raw_next2 = raw_next;
        if (FMT == ANSLIN_FMT_BF16) { raw_next = raw.load(0, lane); raw_next2 = raw.load(1, lane); }
        for (uint32_t u = 0; u < units; ++u) {
          const uint32_t seq = seq0 + u * cnt + idx;
          const uint32_t slot = seq % p.U, lap = seq / p.U;
          const uint32_t slot_a = slots_s + slot * p.slot_bytes;
          for (uint32_t spins = 0; lapw[slot] < lap;) {  // a waiting decoder sleeps: it must not take issue slots
            __nanosleep(100);
            if (++spins > (1u << 24)) __trap();
          }
          mbar_wait<100>(empty_s + 8 * slot, (lap & 1u) ^ 1u);
          if (lane == 0) lapw[slot] = lap + 1u;
          const int k_elem = int(kt * cv.tile_k + u * unit_k_of(FMT));
          if (lane == 0) {
            mbar_arrive_expect_tx(full_s + 8 * slot, xbytes);
            if (p.layout == kLayoutSW32) {
              tma_load_2d(slot_a + kUnitBytes, &tmx, k_elem, 0, full_s + 8 * slot);
            } else {  // two 16-byte-wide boxes = two K-adjacent columns of 8x16B core matrices
              tma_load_2d(slot_a + kUnitBytes, &tmx, k_elem, 0, full_s + 8 * slot);
              tma_load_2d(slot_a + kUnitBytes + p.mpad * 16u, &tmx, k_elem + unit_k_of(FMT) / 2, 0, full_s + 8 * slot);
            }
          }
          SmemEmit emit{slot_a, p.layout};
          const uint32_t *sz_row = nullptr;
          if (FMT == ANSLIN_FMT_INT4_AWQ)
            sz_row = reinterpret_cast<const uint32_t *>(cv.base + cv.off_scales) +
                     size_t(uint32_t(k_elem) / cv.group) * cv.n_out + size_t(stripe) * kTileN;
          decode_unit<FMT, PAYLOAD>(s, smem0 + tab_off, lane, lt, int(u), raw, raw_next, raw_next2, sz_row, emit);
          fence_proxy_async();  // generic-proxy stores -> visible to the tensor core's async proxy
          __syncwarp();
          if (lane == 0) mbar_arrive(full_s + 8 * slot);
        }
      }
      cp_async_wait_all();
    }
  } else if (warp == kMmaWarp) {
    // ===================== MMA issuer: one thread drives the tensor core =====================
    const uint32_t idesc = make_idesc(TR::c, TR::ab, TR::ab, 128, p.mpad);
    uint32_t seq = 0, si = 0;
    for (uint32_t t = t_begin; t < t_end; ++si) {
      const uint32_t ka = t % KT, nt = min(KT - ka, t_end - t), ab = si & 1u;
      mbar_wait<100>(tempty_s + 8 * ab, ((si >> 1) & 1u) ^ 1u);  // epilogue has drained this accumulator
      tc_fence_after();
      const uint32_t n_units = nt * units;
      for (uint32_t j = 0; j < n_units; ++j, ++seq) {
        const uint32_t slot = seq % p.U, par = (seq / p.U) & 1u;
        mbar_wait<40>(full_s + 8 * slot, par);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t a = slots_s + slot * p.slot_bytes, b = a + kUnitBytes;
          uint64_t ad, bd;
          if (p.layout == kLayoutSW32) {
            ad = make_smem_desc(a, 16, 256, kLayoutSW32);
            bd = make_smem_desc(b, 16, 256, kLayoutSW32);
          } else {
            ad = make_smem_desc(a, 2048, 128, kLayoutNone);
            bd = make_smem_desc(b, p.mpad * 16u, 128, kLayoutNone);
          }
          umma<TR::kind>(tmem_base + ab * p.mpad, ad, bd, idesc, j > 0 ? 1u : 0u);
          umma_commit(empty_s + 8 * slot);  // frees the slot when the MMA has read it
          if (j + 1 == n_units) umma_commit(tfull_s + 8 * ab);
        }
        __syncwarp();
      }
      t += nt;
    }
  } else {
    // ===================== epilogue warps 0..3 =====================
    EpiParams ep{p.x_scale, reinterpret_cast<const __half *>(cv.base + cv.off_scales), cv.w_scale, p.y, p.ldy, p.partials,
                 p.counters, p.m, p.mpad};
    epilogue_run<FMT>(ep, tmem_base, tfull_s, tempty_s, flag, t_begin, t_end, KT, G, T, warp, lane);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, p.tmem_cols);
}

// ------------------------------------------------------------------------------------------------
// Dense comparator: same MMA / TMEM / epilogue / split-K scheme, operands by TMA (SWIZZLE_128B).
// ------------------------------------------------------------------------------------------------
struct DenseParams {
  const void *w_scale_h;   // int8: fp16[n_out]
  float w_scale;
  const float *x_scale;
  float *y;
  int64_t ldy;
  uint32_t *partials, *counters;
  uint32_t n_out, k_in, m, mpad, S /*stages*/, stage_bytes, tmem_cols, KB /*k blocks of 128 B*/;
};
constexpr int kDenseThreads = 32 * 6;  // warps 0-3 epilogue, 4 MMA, 5 TMA producer

template <uint32_t FMT>
__global__ void __launch_bounds__(kDenseThreads, 1) dense_gemm_kernel(const __grid_constant__ CUtensorMap tmw,
                                                                       const __grid_constant__ CUtensorMap tmx, DenseParams p) {
  using TR = FmtTraits<FMT>;
  constexpr int KE = 128 / TR::xbytes;           // K elements per 128-byte stage row
  constexpr int UK = 32 / TR::xbytes;            // K elements per MMA
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *smem = smem_raw + (smem0 - smem_u32(smem_raw));
  const uint32_t bar_off = p.S * p.stage_bytes;
  const uint32_t full_s = smem0 + bar_off, empty_s = full_s + 8 * kMaxSlots, tfull_s = empty_s + 8 * kMaxSlots,
                 tempty_s = tfull_s + 16, tmemptr_s = tempty_s + 16;
  volatile uint32_t *tmemptr = reinterpret_cast<volatile uint32_t *>(smem + bar_off + 16 * kMaxSlots + 32);
  volatile uint32_t *flag = reinterpret_cast<volatile uint32_t *>(smem + bar_off + 16 * kMaxSlots + 40);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t G = gridDim.x, KT = p.KB, T = (p.n_out / kTileN) * KT;
  if (threadIdx.x == 0) {
    for (uint32_t i = 0; i < p.S; ++i) { mbar_init(full_s + 8 * i, 1); mbar_init(empty_s + 8 * i, 1); }
    for (uint32_t i = 0; i < 2; ++i) { mbar_init(tfull_s + 8 * i, 1); mbar_init(tempty_s + 8 * i, kEpiWarps); }
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc(tmemptr_s, p.tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmemptr;
  const uint32_t t_begin = cta_first_tile(blockIdx.x, G, T), t_end = cta_first_tile(blockIdx.x + 1, G, T);

  if (warp == 5) {
    if (lane == 0) {
      uint32_t seq = 0;
      for (uint32_t t = t_begin; t < t_end; ++t, ++seq) {
        const uint32_t stripe = t / KT, kb = t % KT, slot = seq % p.S, par = (seq / p.S) & 1u;
        mbar_wait(empty_s + 8 * slot, par ^ 1u);
        const uint32_t a = smem0 + slot * p.stage_bytes;
        mbar_arrive_expect_tx(full_s + 8 * slot, p.stage_bytes);
        tma_load_2d(a, &tmw, int(kb * KE), int(stripe * kTileN), full_s + 8 * slot);
        tma_load_2d(a + 16384, &tmx, int(kb * KE), 0, full_s + 8 * slot);
      }
    }
  } else if (warp == kMmaWarp) {
    const uint32_t idesc = make_idesc(TR::c, TR::ab, TR::ab, 128, p.mpad);
    uint32_t seq = 0, si = 0;
    for (uint32_t t = t_begin; t < t_end; ++si) {
      const uint32_t ka = t % KT, nt = min(KT - ka, t_end - t), ab = si & 1u;
      mbar_wait(tempty_s + 8 * ab, ((si >> 1) & 1u) ^ 1u);
      tc_fence_after();
      for (uint32_t j = 0; j < nt; ++j, ++seq) {
        const uint32_t slot = seq % p.S, par = (seq / p.S) & 1u;
        mbar_wait(full_s + 8 * slot, par);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t a = smem0 + slot * p.stage_bytes, b = a + 16384;
#pragma unroll
          for (int k = 0; k < 4; ++k)
            umma<TR::kind>(tmem_base + ab * p.mpad, make_smem_desc(a + k * 32, 16, 1024, kLayoutSW128),
                           make_smem_desc(b + k * 32, 16, 1024, kLayoutSW128), idesc, (j > 0 || k > 0) ? 1u : 0u);
          umma_commit(empty_s + 8 * slot);
          if (j + 1 == nt) umma_commit(tfull_s + 8 * ab);
        }
        __syncwarp();
      }
      t += nt;
    }
    (void)UK;
  } else {
    EpiParams ep{p.x_scale, reinterpret_cast<const __half *>(p.w_scale_h), p.w_scale, p.y, p.ldy, p.partials, p.counters, p.m, p.mpad};
    epilogue_run<FMT>(ep, tmem_base, tfull_s, tempty_s, flag, t_begin, t_end, KT, G, T, warp, lane);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, p.tmem_cols);
}

// ------------------------------------------------------------------------------------------------
// Host helpers
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

// 2-D row-major tensor [rows x cols] of `ebytes`-byte elements, leading dimension ld elements.
bool make_map_2d(CUtensorMap *map, const void *ptr, int ebytes, uint64_t cols, uint64_t rows, uint64_t ld, uint32_t box_cols,
                 uint32_t box_rows, CUtensorMapSwizzle swz) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows}, strides[1] = {ld * uint64_t(ebytes)};
  cuuint32_t box[2] = {box_cols, box_rows}, estr[2] = {1, 1};
  CUtensorMapDataType dt = ebytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_UINT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8;
  return fn(map, dt, 2, const_cast<void *>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
            CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int num_sms() {
  static int n = [] {
    int dev = 0, v = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    return v;
  }();
  return n;
}

uint32_t mpad_of(int32_t m) { return uint32_t((m + 15) / 16 * 16); }
uint32_t tmem_cols_of(uint32_t mpad) {
  uint32_t c = 32;
  while (c < 2 * mpad) c <<= 1;
  return c;
}
constexpr size_t kSmemMax = 232448;  // 227 KiB opt-in per CTA
// Persistent grid: one CTA per SM, but never fewer than `min_tiles` tiles per CTA (a CTA's decoder
// warps work on that many tiles concurrently, and fewer CTAs per stripe = fewer split-K partials).
uint32_t grid_of(uint32_t n_tiles, uint32_t min_tiles) {
  const uint64_t by_work = std::max<uint64_t>(1, n_tiles / min_tiles);
  return uint32_t(std::min<uint64_t>(by_work, uint64_t(std::max(1, num_sms()))));
}

struct Workspace { size_t counters_off, partials_off, total; };
Workspace workspace_layout(uint32_t stripes, uint32_t grid, uint32_t mpad) {
  Workspace w;
  w.counters_off = 0;
  w.partials_off = align16(size_t(stripes) * 4 + 256);
  w.total = w.partials_off + size_t(grid) * 2 * mpad * kTileN * 4;
  return w;
}

bool x_dtype_ok(uint32_t fmt, uint32_t dt) {
  return (fmt == ANSLIN_FMT_BF16 && dt == ANSLIN_DT_BF16) || (fmt == ANSLIN_FMT_INT4_AWQ && dt == ANSLIN_DT_F16) ||
         (fmt == ANSLIN_FMT_INT8 && dt == ANSLIN_DT_I8) || (fmt == ANSLIN_FMT_FP8_E4M3 && dt == ANSLIN_DT_FP8_E4M3);
}

template <uint32_t FMT, bool PAYLOAD>
int launch_fused(const anslin_weight *w, const CUtensorMap &tmx, GemmParams &p, uint32_t grid, size_t smem, cudaStream_t st) {
  auto kern = fused_gemm_kernel<FMT, PAYLOAD>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess) return ANSLIN_ERR_CUDA;
  kern<<<grid, kGemmThreads, smem, st>>>(tmx, p);
  ++g_launches;
  (void)w;
  if (getenv("ANSLIN_DEBUG")) {  // debugging aid only: synchronous error report
    cudaError_t e = cudaStreamSynchronize(st);
    fprintf(stderr, "[anslin] fused grid=%u smem=%zu D=%u U=%u mpad=%u tiles=%u: %s\n", grid, smem, p.D, p.U, p.mpad,
            p.cv.n_tiles, cudaGetErrorString(e));
  }
  return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}

int gemm_one(const anslin_weight *w, const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m, const void *x_scale_dev,
             void *y_dev, int64_t ldy, void *workspace_dev, size_t workspace_bytes, cudaStream_t st) {
  if (!w || !w->dev || !x_dev || !y_dev || !workspace_dev) return ANSLIN_ERR_INVALID_ARG;
  if (m < 1 || m > 256) return ANSLIN_ERR_UNSUPPORTED;
  const Header &h = w->h;
  if (!x_dtype_ok(h.format, x_dtype)) return ANSLIN_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(x_dev) | reinterpret_cast<uintptr_t>(y_dev) | reinterpret_cast<uintptr_t>(workspace_dev)) & 15)
    return ANSLIN_ERR_INVALID_ARG;
  const bool scaled = h.format == ANSLIN_FMT_INT8 || h.format == ANSLIN_FMT_FP8_E4M3;
  if (scaled && !x_scale_dev) return ANSLIN_ERR_INVALID_ARG;
  const int xb = (h.format == ANSLIN_FMT_BF16 || h.format == ANSLIN_FMT_INT4_AWQ) ? 2 : 1;
  if (ldx < int64_t(h.k_in) || (ldx * xb) % 16 || ldy < int64_t(h.n_out)) return ANSLIN_ERR_INVALID_ARG;
  if (num_sms() <= 0) return ANSLIN_ERR_CUDA;

  GemmParams p;
  p.cv = view_of(w);
  p.m = uint32_t(m);
  p.mpad = mpad_of(m);
  p.slot_bytes = kUnitBytes + p.mpad * 32u;
  p.tmem_cols = tmem_cols_of(p.mpad);
  p.x_scale = static_cast<const float *>(x_scale_dev);
  p.y = static_cast<float *>(y_dev);
  p.ldy = ldy;
  const char *lay = getenv("ANSLIN_LAYOUT");  // debug: "none" selects the unswizzled core-matrix layout
  p.layout = (lay && lay[0] == 'n') ? kLayoutNone : kLayoutSW32;
  uint32_t min_tiles = 12;
  if (const char *e = getenv("ANSLIN_MIN_TILES")) min_tiles = uint32_t(std::max(1, atoi(e)));
  const uint32_t grid = grid_of(h.n_tiles, min_tiles), stripes = h.n_out / kTileN;
  // ring sizing: D decoder warps (1 KiB compressed-word ring each) and U operand slots
  const size_t fixed = 2048 /*align slack*/ + 2048 /*ring alignment*/ + 16384 + 1056 + 16 * kMaxSlots + 64 + 4 * kMaxSlots;
  uint32_t D = kMaxDecWarps, U = 0;
  const char *denv = getenv("ANSLIN_DECODER_WARPS");
  if (denv && atoi(denv) > 0) D = uint32_t(std::min(atoi(denv), kMaxDecWarps));
  if (!getenv("ANSLIN_DMAX")) {  // even rounds: a CTA with tpc tiles needs ceil(tpc/D) tile-times; use the fewest warps that keep that count
    const uint32_t tpc = (h.n_tiles + grid - 1) / grid, rounds = (tpc + D - 1) / D;
    D = std::max(1u, (tpc + rounds - 1) / rounds);
  }
  for (;; --D) {
    const size_t left = kSmemMax - fixed - size_t(D) * kRingBytes;
    U = uint32_t(std::min<size_t>(left / p.slot_bytes, kMaxSlots));
    if (U >= D + 2 || D == 1) break;
  }
  if (U < 2) return ANSLIN_ERR_UNSUPPORTED;
  p.D = D;
  p.U = U;
  const size_t smem = fixed + size_t(D) * kRingBytes + size_t(U) * p.slot_bytes;
  const Workspace ws = workspace_layout(stripes, grid, p.mpad);
  if (workspace_bytes < ws.total) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  p.counters = reinterpret_cast<uint32_t *>(static_cast<uint8_t *>(workspace_dev) + ws.counters_off);
  p.partials = reinterpret_cast<uint32_t *>(static_cast<uint8_t *>(workspace_dev) + ws.partials_off);
  if (cudaMemsetAsync(p.counters, 0, size_t(stripes) * 4, st) != cudaSuccess) return ANSLIN_ERR_CUDA;

  CUtensorMap tmx;
  const uint32_t uk = unit_k_of(h.format);
  const bool ok = p.layout == kLayoutSW32
                      ? make_map_2d(&tmx, x_dev, xb, h.k_in, uint64_t(m), uint64_t(ldx), uk, p.mpad, CU_TENSOR_MAP_SWIZZLE_32B)
                      : make_map_2d(&tmx, x_dev, xb, h.k_in, uint64_t(m), uint64_t(ldx), uk / 2, p.mpad, CU_TENSOR_MAP_SWIZZLE_NONE);
  if (!ok) return ANSLIN_ERR_CUDA;
  const bool pay = h.flags & ANSLIN_FLAG_STATE_PAYLOAD;
  switch (h.format) {
    case ANSLIN_FMT_BF16:
      return pay ? launch_fused<ANSLIN_FMT_BF16, true>(w, tmx, p, grid, smem, st) : launch_fused<ANSLIN_FMT_BF16, false>(w, tmx, p, grid, smem, st);
    case ANSLIN_FMT_FP8_E4M3: return launch_fused<ANSLIN_FMT_FP8_E4M3, false>(w, tmx, p, grid, smem, st);
    case ANSLIN_FMT_INT8: return launch_fused<ANSLIN_FMT_INT8, false>(w, tmx, p, grid, smem, st);
    case ANSLIN_FMT_INT4_AWQ: return launch_fused<ANSLIN_FMT_INT4_AWQ, false>(w, tmx, p, grid, smem, st);
  }
  return ANSLIN_ERR_UNSUPPORTED;
}

template <uint32_t FMT, bool PAYLOAD>
int launch_decode(const ContainerView &cv, void *out, cudaStream_t st) {
  uint32_t per_sm = 4;
  if (const char *e = getenv("ANSLIN_DECODE_CTAS_PER_SM")) per_sm = uint32_t(std::max(1, atoi(e)));  // debug knob
  const uint32_t ctas = std::min<uint32_t>((cv.n_tiles + kDecWarps - 1) / kDecWarps, uint32_t(std::max(1, num_sms())) * per_sm);
  decode_kernel<FMT, PAYLOAD><<<ctas, kDecWarps * 32, 0, st>>>(cv, static_cast<uint8_t *>(out));
  ++g_launches;
  return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}

template <uint32_t FMT>
int launch_dense(const CUtensorMap &tmw, const CUtensorMap &tmx, DenseParams &p, uint32_t grid, size_t smem, cudaStream_t st) {
  auto kern = dense_gemm_kernel<FMT>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess) return ANSLIN_ERR_CUDA;
  kern<<<grid, kDenseThreads, smem, st>>>(tmw, tmx, p);
  ++g_launches;
  return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}

}  // namespace

extern "C" {

int anslin_last_launch_count(void) { return g_launches; }

int anslin_decode(const anslin_weight *w, void *w_out_dev, size_t capacity, void *stream) {
  g_launches = 0;
  if (!w || !w->dev || !w_out_dev) return ANSLIN_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(w_out_dev) & 15) return ANSLIN_ERR_INVALID_ARG;
  const Header &h = w->h;
  const size_t need = h.format == ANSLIN_FMT_BF16 ? size_t(h.n_out) * h.k_in * 2
                      : h.format == ANSLIN_FMT_INT4_AWQ ? size_t(h.n_out) * h.k_in / 2 : size_t(h.n_out) * h.k_in;
  if (capacity < need) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  if (num_sms() <= 0) return ANSLIN_ERR_CUDA;
  const ContainerView cv = view_of(w);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  switch (h.format) {
    case ANSLIN_FMT_BF16:
      return (h.flags & ANSLIN_FLAG_STATE_PAYLOAD) ? launch_decode<ANSLIN_FMT_BF16, true>(cv, w_out_dev, st)
                                                    : launch_decode<ANSLIN_FMT_BF16, false>(cv, w_out_dev, st);
    case ANSLIN_FMT_FP8_E4M3: return launch_decode<ANSLIN_FMT_FP8_E4M3, false>(cv, w_out_dev, st);
    case ANSLIN_FMT_INT8: return launch_decode<ANSLIN_FMT_INT8, false>(cv, w_out_dev, st);
    case ANSLIN_FMT_INT4_AWQ: return launch_decode<ANSLIN_FMT_INT4_AWQ, false>(cv, w_out_dev, st);
  }
  return ANSLIN_ERR_UNSUPPORTED;
}

size_t anslin_gemm_workspace_bytes(const anslin_weight *w, int32_t m) {
  if (!w || m < 1 || m > 256) return 0;
  return workspace_layout(w->h.n_out / kTileN, uint32_t(std::max(1, std::max(num_sms(), 148))), mpad_of(m)).total;
}

int anslin_gemm(const anslin_weight *w, const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m, const void *x_scale_dev,
                void *y_dev, int64_t ldy, void *workspace_dev, size_t workspace_bytes, void *stream) {
  g_launches = 0;
  return gemm_one(w, x_dev, x_dtype, ldx, m, x_scale_dev, y_dev, ldy, workspace_dev, workspace_bytes, static_cast<cudaStream_t>(stream));
}

int anslin_gemm_grouped(const anslin_weight *const *experts, int32_t n_experts, const int32_t *rows_per_expert_host,
                        const void *x_dev, uint32_t x_dtype, int64_t ldx, const void *x_scale_dev, void *y_dev, int64_t ldy,
                        void *workspace_dev, size_t workspace_bytes, void *stream) {
  g_launches = 0;
  if (!experts || n_experts < 1 || !rows_per_expert_host) return ANSLIN_ERR_INVALID_ARG;
  int64_t row = 0;
  for (int e = 0; e < n_experts; ++e) {
    const int32_t rows = rows_per_expert_host[e];
    if (rows < 0 || !experts[e]) return ANSLIN_ERR_INVALID_ARG;
    if (rows == 0) continue;
    const Header &h = experts[e]->h;
    if (h.format != experts[0]->h.format || h.n_out != experts[0]->h.n_out || h.k_in != experts[0]->h.k_in) return ANSLIN_ERR_INVALID_ARG;
    const int xb = (h.format == ANSLIN_FMT_BF16 || h.format == ANSLIN_FMT_INT4_AWQ) ? 2 : 1;
    const uint8_t *xe = static_cast<const uint8_t *>(x_dev) + size_t(row) * ldx * xb;
    const float *xs = x_scale_dev ? static_cast<const float *>(x_scale_dev) + row : nullptr;
    float *ye = static_cast<float *>(y_dev) + size_t(row) * ldy;
    // Y/X row offsets keep 16-byte alignment only if the row pitch does; require it
    if ((reinterpret_cast<uintptr_t>(xe) | reinterpret_cast<uintptr_t>(ye)) & 15) return ANSLIN_ERR_INVALID_ARG;
    int rc = gemm_one(experts[e], xe, x_dtype, ldx, rows, xs, ye, ldy, workspace_dev, workspace_bytes, static_cast<cudaStream_t>(stream));
    if (rc != ANSLIN_OK) return rc;
    row += rows;
  }
  return ANSLIN_OK;
}

size_t anslin_dense_workspace_bytes(uint32_t n_out, uint32_t k_in, int32_t m) {
  (void)k_in;
  if (m < 1 || m > 256 || n_out % kTileN) return 0;
  return workspace_layout(n_out / kTileN, uint32_t(std::max(num_sms(), 148)), mpad_of(m)).total;
}

int anslin_dense_gemm(uint32_t format, const void *w_dev, uint32_t n_out, uint32_t k_in, const void *w_scale_dev, float w_scale,
                      const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m, const void *x_scale_dev, void *y_dev,
                      int64_t ldy, void *workspace_dev, size_t workspace_bytes, void *stream) {
  g_launches = 0;
  if (!w_dev || !x_dev || !y_dev || !workspace_dev) return ANSLIN_ERR_INVALID_ARG;
  if (format > ANSLIN_FMT_INT4_AWQ || m < 1 || m > 256) return ANSLIN_ERR_UNSUPPORTED;
  // the int4 slot takes fp16 weights (what AWQ dequantises to): same MMA kind as the fused int4 path
  const uint32_t xd_need = format == ANSLIN_FMT_INT4_AWQ ? ANSLIN_DT_F16 : 0;
  if (format == ANSLIN_FMT_INT4_AWQ ? x_dtype != xd_need : !x_dtype_ok(format, x_dtype)) return ANSLIN_ERR_INVALID_ARG;
  const int xb = (format == ANSLIN_FMT_BF16 || format == ANSLIN_FMT_INT4_AWQ) ? 2 : 1;
  const uint32_t ke = 128 / xb;
  if (n_out % kTileN || k_in % ke) return ANSLIN_ERR_UNSUPPORTED;
  if ((reinterpret_cast<uintptr_t>(w_dev) | reinterpret_cast<uintptr_t>(x_dev) | reinterpret_cast<uintptr_t>(y_dev) |
       reinterpret_cast<uintptr_t>(workspace_dev)) & 15)
    return ANSLIN_ERR_INVALID_ARG;
  const bool scaled = format == ANSLIN_FMT_INT8 || format == ANSLIN_FMT_FP8_E4M3;
  if (scaled && !x_scale_dev) return ANSLIN_ERR_INVALID_ARG;
  if (format == ANSLIN_FMT_INT8 && !w_scale_dev) return ANSLIN_ERR_INVALID_ARG;
  if (num_sms() <= 0) return ANSLIN_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  DenseParams p;
  p.w_scale_h = w_scale_dev; p.w_scale = w_scale; p.x_scale = static_cast<const float *>(x_scale_dev);
  p.y = static_cast<float *>(y_dev); p.ldy = ldy; p.n_out = n_out; p.k_in = k_in; p.m = uint32_t(m); p.mpad = mpad_of(m);
  p.KB = k_in / ke;
  p.stage_bytes = 16384 + p.mpad * 128u;
  p.tmem_cols = tmem_cols_of(p.mpad);
  const size_t fixed = 1024 + 16 * kMaxSlots + 64;
  p.S = uint32_t(std::min<size_t>((kSmemMax - fixed) / p.stage_bytes, 12));
  const size_t smem = fixed + size_t(p.S) * p.stage_bytes;
  const uint32_t stripes = n_out / kTileN, T = stripes * p.KB, grid = grid_of(T, 8);
  const Workspace ws = workspace_layout(stripes, grid, p.mpad);
  if (workspace_bytes < ws.total) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  p.counters = reinterpret_cast<uint32_t *>(static_cast<uint8_t *>(workspace_dev) + ws.counters_off);
  p.partials = reinterpret_cast<uint32_t *>(static_cast<uint8_t *>(workspace_dev) + ws.partials_off);
  if (cudaMemsetAsync(p.counters, 0, size_t(stripes) * 4, st) != cudaSuccess) return ANSLIN_ERR_CUDA;
  CUtensorMap tmw, tmx;
  if (!make_map_2d(&tmw, w_dev, xb, k_in, n_out, k_in, ke, kTileN, CU_TENSOR_MAP_SWIZZLE_128B)) return ANSLIN_ERR_CUDA;
  if (!make_map_2d(&tmx, x_dev, xb, k_in, uint64_t(m), uint64_t(ldx), ke, p.mpad, CU_TENSOR_MAP_SWIZZLE_128B)) return ANSLIN_ERR_CUDA;
  switch (format) {
    case ANSLIN_FMT_BF16: return launch_dense<ANSLIN_FMT_BF16>(tmw, tmx, p, grid, smem, st);
    case ANSLIN_FMT_INT4_AWQ: return launch_dense<ANSLIN_FMT_INT4_AWQ>(tmw, tmx, p, grid, smem, st);
    case ANSLIN_FMT_FP8_E4M3: return launch_dense<ANSLIN_FMT_FP8_E4M3>(tmw, tmx, p, grid, smem, st);
    case ANSLIN_FMT_INT8: return launch_dense<ANSLIN_FMT_INT8>(tmw, tmx, p, grid, smem, st);
  }
  return ANSLIN_ERR_UNSUPPORTED;
}

}  // extern "C"
