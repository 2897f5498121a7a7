// libanslin device side (sm_100a): the decode-only kernels, the two fused rANS-decode + tcgen05 GEMM kernels, the dense
// tcgen05 comparator, and their C-ABI launchers.
//
// Decode only (anslin_decode): decode_lanes_kernel (decode_lanes.cuh) for lane-stream containers with 32-row tiles — decoded
//   rows leave through TMA stores — and decode_kernel (below) for every other layout.
//
// Fused kernel = Alg V.1 (P:l.196-252) re-designed for Blackwell:
//   * fused_tmem_kernel (fused_tmem.cuh): lane-stream containers with 32-row tiles.  Teams of four decoder warps hand the
//     decoded operand to the tensor core through TENSOR MEMORY (tcgen05.st -> tcgen05.mma with A in TMEM); one issuer warp
//     per team issues the MMAs and the TMA loads of the X slices; stream-K split over teams; a work item is a pair of
//     k-tiles (two chains per warp) or, in launches with at most one tile per team, a single k-tile.  The path bench.py times.
//   * fused_gemm_kernel (below): every other container layout, batches above 96 rows, and launches of few, long tile pairs.
//     The paper's single producer warp becomes up to 16 decoder warps per CTA (decode is the bottleneck at small batch,
//     P:l.306), the consumer warps become ONE thread issuing tcgen05.mma with the accumulator in TMEM; ready[2] flags
//     (P:l.210) become mbarrier full/empty pairs over private slots of 4 KiB operand units (128 rows x 32 B = one MMA K
//     step) in shared memory ("ring buffer lets decode run several sub-tiles ahead", P:l.297); activations arrive by
//     TMA (cp.async.bulk.tensor) into the same slot.
//   In both, the weights are the MMA "A" operand (M = 128 weight rows) and the batch is MMA N.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <type_traits>
#include <atomic>
#include <chrono>

#include "anslin_internal.h"
#include "decode_core.cuh"

using namespace anslin;


namespace {


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
#ifndef ANSLIN_WAIT_HINT
#define ANSLIN_WAIT_HINT 1000000
#endif
// Bounded, blocking wait: mbarrier.try_wait suspends the warp in hardware for up to the time hint, so a
// waiting warp (MMA issuer, epilogue, slot-starved decoder) takes no issue slots from the decoder warps
// that share its scheduler.  A protocol bug traps (launch failure) instead of hanging the GPU.
template <int kUnused = 0>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0, tries = 0;
  while (true) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity), "r"(uint32_t(ANSLIN_WAIT_HINT))
        : "memory");
    if (done) break;
    if (++tries > (1u << 22)) __trap();
  }
}
// Programmatic dependent launch: the next kernel of the stream may start (prologue, table build, tile fetch: weights
// only) while this one drains; everything that depends on the previous kernel (X, scales, Y, workspace) is touched
// only after grid_dep_wait().
__device__ __forceinline__ void grid_dep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
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
__device__ __forceinline__ void named_bar_arrive(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// non-blocking probe of an mbarrier phase
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(done)
      : "r"(bar), "r"(parity)
      : "memory");
  return done != 0;
}
// named barriers 2 and 3: MMA warp -> epilogue warps, "accumulator of segment si is complete".  The id alternates with the
// segment: a second arrive on the same id then belongs to segment si + 2, which the MMA warp reaches only after the
// epilogue warps have drained segment si (tempty), i.e. after all four have passed the barrier for it.
constexpr int kBarEpiGo = 2;
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
template <> struct FmtTraits<ANSLIN_FMT_BF16_PAIR4> : FmtTraits<ANSLIN_FMT_BF16> {};
template <> struct FmtTraits<ANSLIN_FMT_INT4_AWQ> { static constexpr int kind = 0; static constexpr uint32_t c = 1, ab = 0; static constexpr int xbytes = 2; };
template <> struct FmtTraits<ANSLIN_FMT_FP8_E4M3> { static constexpr int kind = 1; static constexpr uint32_t c = 1, ab = 0; static constexpr int xbytes = 1; };
template <> struct FmtTraits<ANSLIN_FMT_FP4_E2M1> { static constexpr int kind = 1; static constexpr uint32_t c = 1, ab = 0; static constexpr int xbytes = 1; };
template <> struct FmtTraits<ANSLIN_FMT_INT8> { static constexpr int kind = 2; static constexpr uint32_t c = 2, ab = 1; static constexpr int xbytes = 1; };

// ------------------------------------------------------------------------------------------------
// Parameters
// ------------------------------------------------------------------------------------------------
struct ContainerView {
  const uint8_t *base;
  uint64_t off_freq, off_offsets, off_records, off_raw, off_scales, total;
  uint32_t n_out, k_in, tile_n, tile_k, KT, n_tiles, units, group, flags, max_seg_bytes;
  float w_scale;
};

ContainerView view_of(const anslin_weight *w) {
  const Header &h = w->h;
  ContainerView v;
  v.base = w->dev;
  v.off_freq = h.off_freq; v.off_offsets = h.off_offsets; v.off_records = h.off_records; v.off_raw = h.off_raw;
  v.off_scales = h.format == ANSLIN_FMT_BF16_PAIR4 ? h.off_zeros /* the 16-byte exponent code table */ : h.off_scales; v.total = h.total_bytes;
  v.n_out = h.n_out; v.k_in = h.k_in; v.tile_n = h.tile_n; v.tile_k = h.tile_k; v.KT = h.k_in / h.tile_k; v.n_tiles = h.n_tiles;
  v.units = h.tile_k / unit_k_of(h.format); v.group = h.group_size; v.flags = h.flags; v.w_scale = h.w_scale;
  v.max_seg_bytes = h.max_seg_bytes;
  return v;
}

// A warp decodes J tiles at once (decode_core.cuh).  RB = tile_n / 32; a 128-row MMA unit is filled by
// NW warps: 32-row tiles: J in {1, 2, 4}, NW = 4 / J; 128-row tiles: J = 1, NW = 1.
template <int RB, int J> struct TileTraits {
  static_assert((RB == 1 && (J == 1 || J == 2 || J == 4)) || (RB == 4 && J == 1), "unsupported tile / interleave combination");
  static constexpr int Q = 4 / RB /*tiles per (stripe, k-tile) group*/, NW = Q / J /*warps per unit*/;
};
#ifndef ANSLIN_J32
#define ANSLIN_J32 2
#endif
// Most decoder warps a CTA may have.  16 (+ 5 = 672 threads) lets ptxas use up to 96 registers per thread; with 20 the cap
// is 80 and the decode loop's schedule gets tighter: 20 was never faster (M = 1 .. 75) and 3 % slower at M = 75.
#ifndef ANSLIN_MAXDEC
#define ANSLIN_MAXDEC 16
#endif
constexpr int kJ32 = ANSLIN_J32;   // tiles a warp interleaves when tiles have 32 rows

__host__ __device__ constexpr size_t row_bytes_of(uint32_t fmt, size_t k) {
  return is_bf16_like(fmt) ? k * 2 : is_packed4(fmt) ? k / 2 : k;
}

// ------------------------------------------------------------------------------------------------
// Decode-only kernel (anslin_decode): one warp per J tiles, output row-major W to HBM.
// ------------------------------------------------------------------------------------------------
template <uint32_t FMT, int RB, int J>
struct GlobalEmit {
  static constexpr bool kOperand = false;
  // 32-row tiles (lane = row): a lane's 16-byte chunks of two consecutive units (64 B of its row) are staged in
  // shared memory and written out as 64-byte row segments, 8 rows per store instruction, instead of one 16-byte
  // store per lane into 32 different rows (which bound the kernel at a third of the decoder's rate).
  static constexpr bool kStaged = RB == 1 && !is_packed4(FMT);
  static constexpr uint32_t kStageBytes = kStaged ? 2048 : 0;   // per stream
  uint8_t *tile_out[J];  // &W[first row of tile j][k0] in bytes
  size_t row_bytes;      // bytes per W row
  uint32_t stage;        // shared address of this warp's J staging areas
  int u;
  __device__ __forceinline__ void chunk(int j, int g, int lane, uint4 v) const {  // bf16 / fp8 / int8: 16 B of row-major W
    if constexpr (kStaged) {
      const uint32_t c = uint32_t((u & 1) * 2 + g);
      sts128(stage + uint32_t(j) * kStageBytes + uint32_t(lane) * 64u + ((c ^ ((uint32_t(lane) >> 1) & 3u)) << 4), v);
    } else {
      uint8_t *p = tile_out[j] + size_t((g % RB) * 32 + lane) * row_bytes + size_t(u) * 32 + (g / RB) * 16;
      *reinterpret_cast<uint4 *>(p) = v;
    }
  }
  // after every unit; with staging, units 2n and 2n+1 are flushed together
  __device__ __forceinline__ void unit_done(int lane) const {
    if constexpr (kStaged) {
      if ((u & 1) == 0) return;
      __syncwarp();
#pragma unroll
      for (int j = 0; j < J; ++j)
#pragma unroll
        for (int it = 0; it < 4; ++it) {
          const uint32_t r = uint32_t(it * 8 + (lane >> 2)), c = uint32_t(lane & 3);
          uint4 v;
          asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                       : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                       : "r"(stage + uint32_t(j) * kStageBytes + r * 64u + ((c ^ ((r >> 1) & 3u)) << 4)));
          *reinterpret_cast<uint4 *>(tile_out[j] + size_t(r) * row_bytes + size_t(u - 1) * 32 + c * 16) = v;
        }
      __syncwarp();
    }
  }
  __device__ __forceinline__ void packed(int j, int g, int lane, uint32_t b) const {  // int4: 4 packed bytes = 8 weights
    uint8_t *p = tile_out[j] + size_t((g % RB) * 32 + lane) * row_bytes + size_t(u) * 8 + (g / RB) * 4;
    *reinterpret_cast<uint32_t *>(p) = b;
  }
  __device__ __forceinline__ void packed8(int j, int g, int lane, uint32_t b0, uint32_t b1) const {  // fp4: 8 packed bytes = 16 weights
    uint8_t *p = tile_out[j] + size_t((g % RB) * 32 + lane) * row_bytes + size_t(u) * 16 + (g / RB) * 8;
    *reinterpret_cast<uint2 *>(p) = make_uint2(b0, b1);
  }
};

constexpr int kDecWarps = 8;

// steps of one lane per operand unit of a 32-row tile (lane = row)
__host__ __device__ constexpr int unit_steps32(uint32_t fmt) { return 2 * spc_of(fmt); }

template <uint32_t FMT, int RB, int J, bool PAYLOAD, bool LS>
__global__ void __launch_bounds__(kDecWarps * 32, 2) decode_kernel(ContainerView cv, uint8_t *out, uint32_t stream_bytes) {
  using POL = typename std::conditional<LS, LaneWords, InterleavedWords>::type;
  constexpr int Q = TileTraits<RB, J>::Q;
  extern __shared__ __align__(16) uint8_t dsm[];
  uint32_t *tab = reinterpret_cast<uint32_t *>(dsm);
  uint32_t *cum = tab + kM;
  uint8_t *rings = dsm + 4 * kM + 1056;
  build_slot_table(tab, cum, reinterpret_cast<const uint16_t *>(cv.base + cv.off_freq));
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t ring_s = smem_u32(rings) + uint32_t(warp) * J * stream_bytes;
  const uint32_t stage_s = smem_u32(rings) + uint32_t(kDecWarps) * J * stream_bytes + uint32_t(warp) * J * GlobalEmit<FMT, RB, J>::kStageBytes;
  const uint32_t aux = LS ? ((lane & 1) ? uint32_t(-2) : 2u) : lanemask_lt();
  const uint32_t *offs = reinterpret_cast<const uint32_t *>(cv.base + cv.off_offsets);
  PairLut plut{0, 0, 0, 0};
  if constexpr (FMT == ANSLIN_FMT_BF16_PAIR4) {
    const uint4 c = *reinterpret_cast<const uint4 *>(cv.base + cv.off_scales);
    plut = PairLut{c.x, c.y, c.z, c.w};
  }
  const size_t row_bytes = row_bytes_of(FMT, cv.k_in), tile_row_bytes = row_bytes_of(FMT, cv.tile_k);
  const size_t rtb = raw_tile_bytes(32 * RB, cv.tile_k, PAYLOAD ? ANSLIN_FLAG_STATE_PAYLOAD : 0);
  const int V = int(cv.units) * RB;
  constexpr uint32_t kUnitsPerSeg = LS ? seg_steps_of(FMT) / unit_steps32(FMT) : 1;
  for (uint32_t job = blockIdx.x * kDecWarps + warp; job < cv.n_tiles / J; job += gridDim.x * kDecWarps) {
    typename POL::S s[J];
    RawReader<PAYLOAD> raw[J];
    const uint32_t *sz[J];
    GlobalEmit<FMT, RB, J> emit;
    emit.row_bytes = row_bytes;
    emit.stage = stage_s;
    stream_drain();
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const uint32_t t = job * J + j, grp = t / Q, q = t % Q, stripe = grp / cv.KT, kt = grp % cv.KT;
      const uint8_t *rec = cv.base + cv.off_records + size_t(offs[t]) * 16;
      if constexpr (LS) lane_open(s[j], rec, int(cv.units / kUnitsPerSeg), lane);
      else stream_open(s[j], rec, ring_s + j * stream_bytes, lane);
      emit.tile_out[j] = out + (size_t(stripe) * kTileN + size_t(q) * 32 * RB) * row_bytes + size_t(kt) * tile_row_bytes;
      if (is_bf16_like(FMT)) raw[j].open(cv.base + cv.off_raw + size_t(t) * rtb, V, lane);
      sz[j] = nullptr;
    }
    for (uint32_t u = 0; u < cv.units; ++u) {
      emit.u = int(u);
      if constexpr (LS) {
        if (u % kUnitsPerSeg == 0) {
          lane_open_segments<J>(s, ring_s, stream_bytes, int(u / kUnitsPerSeg), lane);
        }
      }
      decode_unit<FMT, RB, J, PAYLOAD, POL>(s, ring_s, smem_u32(tab), lane, aux, int(u), V, raw, sz, emit, plut);
      emit.unit_done(lane);
    }
  }
  cp_async_wait_all();
}

// ------------------------------------------------------------------------------------------------
// Work split and epilogue helpers shared by the fused and the dense kernel
// ------------------------------------------------------------------------------------------------
constexpr int kEpiWarps = 4;
constexpr int kMmaWarp = 4;
constexpr int kFirstDecWarp = 5;
constexpr int kMaxDecWarps = ANSLIN_MAXDEC;
constexpr int kGemmThreads = 32 * (kFirstDecWarp + kMaxDecWarps);
constexpr int kMaxSlots = 48;

// Work of CTA c (of G): groups [first(c), first(c+1)) of the stripe-major sequence of T (stripe, k-tile)
// groups (stream-K style equal split): a CTA owns at most two partial stripes plus whole stripes.
__host__ __device__ __forceinline__ uint32_t cta_first_tile(uint32_t c, uint32_t G, uint32_t T) { return uint32_t(uint64_t(c) * T / G); }
__host__ __device__ __forceinline__ uint32_t cta_of_tile(uint32_t t, uint32_t G, uint32_t T) {  // largest c with first(c) <= t
  return uint32_t((uint64_t(t + 1) * G + T - 1) / T) - 1;
}

template <uint32_t FMT>
__device__ __forceinline__ float finalize(uint32_t bits, float xs, float ws) {
  if constexpr (FMT == ANSLIN_FMT_INT8) return float(int32_t(bits)) * xs * ws;
  else if constexpr (is_fp8_path(FMT)) return __uint_as_float(bits) * xs * ws;
  else return __uint_as_float(bits);
}
template <uint32_t FMT>
__device__ __forceinline__ uint32_t acc_add(uint32_t a, uint32_t b) {
  if constexpr (FMT == ANSLIN_FMT_INT8) return uint32_t(int32_t(a) + int32_t(b));
  else return __float_as_uint(__uint_as_float(a) + __uint_as_float(b));
}

struct EpiParams {
  const float *x_scale;     // int8 / fp8: f32[m]
  const __half *w_scale_h;  // int8: fp16[n_out]
  float w_scale;            // fp8
  float *y;
  int64_t ldy;
  uint32_t *partials;              // [2*G][mpad][128] raw accumulator bits
  unsigned long long *counters;    // split-K flags, u32 [2 * CTAs of the problem]: flag[c * 2 + seg] = launch epoch once CTA c's partial `seg` is stored
  uint32_t epoch;                  // unique per launch: stale counter contents (any bytes) read as "nobody arrived"
  uint32_t m, mpad;
};
// A stripe whose last split-K contributor is this CTA (shared memory; at most the first and the last segment).
struct FinSeg { uint32_t valid, stripe, c_first, c_last; };

__device__ __forceinline__ uint4 ldcg128(const uint32_t *p) {
  uint4 r;
  asm volatile("ld.global.cg.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

// Epilogue (a10), warps 0..3: TMEM -> registers -> Y for whole stripes, or -> split-K partial.  The CTA
// that contributes LAST to a stripe (global counter) records it in fin[]; splitk_fixup sums it up later.
// YB: Y holds bf16 (the fp32 result rounded to nearest even) instead of f32; a template parameter, so that the f32 kernels'
// code is exactly what it was (a run-time branch here cost the whole kernel 3 % through register allocation).
template <uint32_t FMT, bool YB = false>
__device__ __forceinline__ void epilogue_run(const EpiParams &p, uint32_t tmem_base, uint32_t tfull_s, uint32_t tempty_s,
                                             FinSeg *fin, uint32_t t_begin, uint32_t t_end, uint32_t KT, uint32_t c, uint32_t G,
                                             uint32_t T, int warp, int lane) {
  constexpr bool kScaled = FMT == ANSLIN_FMT_INT8 || is_fp8_path(FMT);
  const uint32_t row = uint32_t(warp * 32 + lane);
  uint32_t si = 0;
  for (uint32_t t = t_begin; t < t_end; ++si) {
    const uint32_t stripe = t / KT, ka = t % KT, nt = min(KT - ka, t_end - t), ab = si & 1u;
    const bool whole = (ka == 0 && nt == KT);
    const uint32_t n = stripe * kTileN + row;
    float ws = 1.0f;
    if (FMT == ANSLIN_FMT_INT8) ws = __half2float(p.w_scale_h[n]);
    if (is_fp8_path(FMT)) ws = p.w_scale;
    // The MMA warp watches the accumulator's mbarrier and releases us through a named barrier: the four
    // epilogue warps sleep in hardware meanwhile instead of polling next to the decoder warps.
    named_bar_sync(kBarEpiGo + int(si & 1u), (kEpiWarps + 1) * 32);
    tc_fence_after();
    const uint32_t seg = (t == t_begin ? 0u : 1u);
    uint32_t *part = p.partials + size_t(c * 2u + seg) * p.mpad * kTileN;
    for (uint32_t c0 = 0; c0 < p.mpad; c0 += 16) {
      uint32_t v[16];
      tmem_ld16(tmem_base + ((uint32_t(warp) * 32u) << 16) + ab * p.mpad + c0, v);
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const uint32_t mm = c0 + j;
        if (mm < p.m) {
          if (whole) {
            const float f = finalize<FMT>(v[j], kScaled ? p.x_scale[mm] : 1.0f, ws);
            if constexpr (YB) reinterpret_cast<__nv_bfloat16 *>(p.y)[size_t(mm) * p.ldy + n] = __float2bfloat16_rn(f);
            else p.y[size_t(mm) * p.ldy + n] = f;
          }
          else part[size_t(mm) * kTileN + row] = v[j];
        }
      }
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(tempty_s + 8 * ab);
    if (!whole) {
      __threadfence();
      named_bar_sync(1, kEpiWarps * 32);
      if (warp == 0) {
        // every thread's partial stores are fenced and the warps have met: raise this segment's flags, one word per reader
        // (flag[(c * 2 + seg) * KT + reader's index among the stripe's contributors]).  The contributors of a stripe are the
        // CTAs c_first .. c_last that hold its k-tiles (known from the shape alone); EVERY one of them sums its own slice of
        // the stripe's outputs once it has seen the flags addressed to it carry this launch's epoch (splitk_fixup): no
        // atomics, no retries under contention, and stale or uninitialised workspace bytes never match the epoch.
        const uint32_t c_first = cta_of_tile(stripe * KT, G, T), c_last = cta_of_tile(stripe * KT + KT - 1, G, T);
        uint32_t *flag = reinterpret_cast<uint32_t *>(p.counters) + size_t(c * 2u + seg) * KT;
        for (uint32_t r = uint32_t(lane); r <= c_last - c_first; r += 32)
          asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(flag + r), "r"(p.epoch) : "memory");
        if (lane == 0) { fin[seg].stripe = stripe; fin[seg].c_first = c_first; fin[seg].c_last = c_last; fin[seg].valid = 1u; }
      }
    }
    t += nt;
  }
}

// Deterministic split-K fix-up by ALL threads of the CTA (call after a CTA-wide barrier that follows
// epilogue_run): for each stripe recorded in fin[] (every stripe this CTA holds a partial of), sum THIS CTA's slice of the
// stripe's outputs over the partials of all contributors in CTA order (bit-reproducible), apply the scales and store Y.
// One item = one batch row x 4 output channels; 16-byte loads, up to 8 contributors in flight per thread.  (One owner CTA
// summing a whole stripe took ~15 us at the end of every launch.)
template <uint32_t FMT, bool YB = false>
__device__ __forceinline__ void splitk_fixup(const EpiParams &p, const FinSeg *fin, uint32_t KT, uint32_t c, uint32_t G, uint32_t T) {   // c: this CTA's index in its problem
  constexpr bool kScaled = FMT == ANSLIN_FMT_INT8 || is_fp8_path(FMT);
  constexpr int kItems = 2;   // items per thread and pass: their loads are all issued before the first add
  for (int seg = 0; seg < 2; ++seg) {
    if (!fin[seg].valid) continue;
    const uint32_t stripe = fin[seg].stripe, c_first = fin[seg].c_first, c_last = fin[seg].c_last;
    // contributor cc's partial slot: its first segment (slot 0) unless the stripe is its second one, which can only
    // be the case for the first contributor (every later one starts inside the stripe)
    const uint32_t first_slot = cta_first_tile(c_first, G, T) < stripe * KT ? 1u : 0u;
    // wait for the flags the contributors address to this CTA (all CTAs of the persistent grid are resident and raise their
    // flags before they get here): one flag per thread
    const uint32_t count = c_last - c_first + 1u, my_index = c - c_first;
    for (uint32_t cc = c_first + threadIdx.x; cc <= c_last; cc += blockDim.x) {
      const uint32_t *flag = reinterpret_cast<const uint32_t *>(p.counters) + size_t(cc * 2u + (cc == c_first ? first_slot : 0u)) * KT + my_index;
      uint32_t v, spins = 0;
      while (true) {
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory");
        if (v == p.epoch) break;
        __nanosleep(64);
        if (++spins > (1u << 24)) __trap();   // a protocol bug traps instead of hanging the GPU
      }
      // consumed: clear the flag, so that a replay of this very launch (CUDA graph: same epoch) starts from "not stored"
      *const_cast<volatile uint32_t *>(flag) = 0u;
    }
    __syncthreads();
    const size_t slot_words = size_t(p.mpad) * kTileN;
    const uint32_t all_items = p.m * 32u, it_begin = my_index * all_items / count, n_items = (my_index + 1u) * all_items / count;
    for (uint32_t it0 = it_begin + threadIdx.x; it0 < n_items; it0 += blockDim.x * kItems) {
      uint32_t acc[kItems][4];
#pragma unroll
      for (int q = 0; q < kItems; ++q)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[q][j] = FMT == ANSLIN_FMT_INT8 ? 0u : __float_as_uint(0.0f);
      for (uint32_t cb = c_first; cb <= c_last; cb += 4) {
        uint4 v[kItems][4];
#pragma unroll
        for (int q = 0; q < kItems; ++q) {
          const uint32_t it = it0 + q * blockDim.x, mm = it >> 5, r4 = (it & 31u) * 4u;
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint32_t cc = cb + j;
            v[q][j] = make_uint4(0, 0, 0, 0);
            if (cc <= c_last && it < n_items) {
              const uint32_t ps = cc * 2u + (cc == c_first ? first_slot : 0u);
              v[q][j] = ldcg128(p.partials + size_t(ps) * slot_words + size_t(mm) * kTileN + r4);
            }
          }
        }
#pragma unroll
        for (int q = 0; q < kItems; ++q)
#pragma unroll
          for (int j = 0; j < 4; ++j) {  // fixed CTA order -> bit-reproducible sums
            acc[q][0] = acc_add<FMT>(acc[q][0], v[q][j].x); acc[q][1] = acc_add<FMT>(acc[q][1], v[q][j].y);
            acc[q][2] = acc_add<FMT>(acc[q][2], v[q][j].z); acc[q][3] = acc_add<FMT>(acc[q][3], v[q][j].w);
          }
      }
#pragma unroll
      for (int q = 0; q < kItems; ++q) {
        const uint32_t it = it0 + q * blockDim.x, mm = it >> 5, n4 = stripe * kTileN + (it & 31u) * 4u;
        if (it >= n_items) continue;
        const float xs = kScaled ? p.x_scale[mm] : 1.0f;
        float o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          float ws = 1.0f;
          if (FMT == ANSLIN_FMT_INT8) ws = __half2float(p.w_scale_h[n4 + j]);
          if (is_fp8_path(FMT)) ws = p.w_scale;
          o[j] = finalize<FMT>(acc[q][j], xs, ws);
        }
        if constexpr (YB) {
          __nv_bfloat16 *yb = reinterpret_cast<__nv_bfloat16 *>(p.y) + size_t(mm) * p.ldy + n4;
          const __nv_bfloat162 lo = __floats2bfloat162_rn(o[0], o[1]), hi = __floats2bfloat162_rn(o[2], o[3]);
          if ((reinterpret_cast<uintptr_t>(yb) & 7) == 0)
            *reinterpret_cast<uint2 *>(yb) = make_uint2(*reinterpret_cast<const uint32_t *>(&lo), *reinterpret_cast<const uint32_t *>(&hi));
          else { yb[0] = lo.x; yb[1] = lo.y; yb[2] = hi.x; yb[3] = hi.y; }
          continue;
        }
        float *yo = p.y + size_t(mm) * p.ldy + n4;
        if ((reinterpret_cast<uintptr_t>(yo) & 15) == 0) *reinterpret_cast<float4 *>(yo) = make_float4(o[0], o[1], o[2], o[3]);
        else { yo[0] = o[0]; yo[1] = o[1]; yo[2] = o[2]; yo[3] = o[3]; }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Fused decode + GEMM kernel
// ------------------------------------------------------------------------------------------------
constexpr int kMaxProblems = 8;
// One GEMM of a launch.  A launch is the concatenation of independent sub-grids: problem i owns CTAs
// [cta0, cta0 + ncta) (grouped MoE experts, or projections that share an input).
struct Problem {
  ContainerView cv;
  const float *x_scale;    // int8 / fp8: f32[m]
  float *y;
  int64_t ldy;
  uint32_t *partials;      // [2*ncta][mpad][128] raw accumulator bits
  unsigned long long *counters;   // [stripes]
  uint32_t m, mpad, cta0, ncta;
};
struct FusedParams {
  Problem prob[kMaxProblems];
  uint32_t nprob;
  uint32_t U, D, B;        // operand slots (= teams * B), decoder warps, slots per team (>= 2)
  uint32_t epoch;          // launch id for the split-K counters
  uint32_t stream_bytes;   // shared memory per stream: word ring + mirror, or the largest staged lane-stream segment
  uint32_t slot_bytes;     // 4096 + max mpad * 32
  uint32_t tmem_cols;
  uint32_t afmt, bfmt;     // tcgen05 a/b format codes (fp8: 0 = e4m3, 1 = e5m2, chosen at run time)
};
struct TensorMaps { CUtensorMap m[kMaxProblems]; };

// Shared-memory unit slot writer: the decoded 16-byte chunk goes where the UMMA K-major SWIZZLE_32B
// canonical layout expects it (P:l.151 "consumed by the GEMM kernel in its required swizzled layout").
template <int RB, int J>
struct SmemEmit {
  static constexpr bool kOperand = true;
  uint32_t slot_a;       // shared address of the unit's A operand (4 KiB)
  uint32_t row0[J];      // first stripe row of stream j's tile
  __device__ __forceinline__ void chunk(int j, int g, int lane, uint4 v) const {
    const uint32_t row = row0[j] + uint32_t((g % RB) * 32 + lane), c = uint32_t(g / RB);
    sts128(slot_a + row * 32u + ((c ^ ((uint32_t(lane) >> 2) & 1u)) << 4), v);  // Swizzle<1,4,3>
  }
  __device__ __forceinline__ void packed(int, int, int, uint32_t) const {}
  __device__ __forceinline__ void packed8(int, int, int, uint32_t, uint32_t) const {}
};

#include "fused_tmem.cuh"
#include "decode_lanes.cuh"

template <uint32_t FMT, int RB, int J, bool PAYLOAD, bool LS, bool YB>
__global__ void __launch_bounds__(kGemmThreads, 1) fused_gemm_kernel(const __grid_constant__ TensorMaps tms,
                                                                      const __grid_constant__ FusedParams P) {
  using TR = FmtTraits<FMT>;
  using POL = typename std::conditional<LS, LaneWords, InterleavedWords>::type;
  constexpr int NW = TileTraits<RB, J>::NW, Q = TileTraits<RB, J>::Q;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 2047u) & ~2047u;
  uint8_t *smem = smem_raw + (smem0 - smem_u32(smem_raw));
  grid_dep_launch_dependents();
  // which problem does this CTA belong to?
  uint32_t pi = 0;
  while (pi + 1 < P.nprob && blockIdx.x >= P.prob[pi + 1].cta0) ++pi;
  const Problem &pr = P.prob[pi];
  const ContainerView &cv = pr.cv;
  const uint32_t c = blockIdx.x - pr.cta0, G = pr.ncta, KT = cv.KT, T = (cv.n_out / kTileN) * KT;
  const uint32_t mpad = pr.mpad, units = cv.units;
  // carve-up
  const uint32_t slots_s = smem0;
  const uint32_t ring_off = P.U * P.slot_bytes;
  const uint32_t tab_off = ring_off + P.D * J * P.stream_bytes;
  uint32_t *tab = reinterpret_cast<uint32_t *>(smem + tab_off);
  uint32_t *cum = reinterpret_cast<uint32_t *>(smem + tab_off + 16384);
  const uint32_t bar_off = tab_off + 16384 + 1056;
  const uint32_t full_s = smem0 + bar_off, empty_s = full_s + 8 * kMaxSlots, tfull_s = empty_s + 8 * kMaxSlots,
                 tempty_s = tfull_s + 16, tmemptr_s = tempty_s + 16;
  volatile uint32_t *tmemptr = reinterpret_cast<volatile uint32_t *>(smem + bar_off + 16 * kMaxSlots + 32);
  FinSeg *fin = reinterpret_cast<FinSeg *>(smem + bar_off + 16 * kMaxSlots + 48);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

  if (threadIdx.x == 0) {
    for (uint32_t i = 0; i < P.U; ++i) { mbar_init(full_s + 8 * i, NW + 1); mbar_init(empty_s + 8 * i, 1); }
    for (uint32_t i = 0; i < 2; ++i) { mbar_init(tfull_s + 8 * i, 1); mbar_init(tempty_s + 8 * i, kEpiWarps); fin[i].valid = 0; }
    fence_mbar_init();
  }
  if (warp == int(P.D) + kEpiWarps) tmem_alloc(tmemptr_s, P.tmem_cols);
  tc_fence_before();
  build_slot_table(tab, cum, reinterpret_cast<const uint16_t *>(cv.base + cv.off_freq));  // ends with __syncthreads()
  tc_fence_after();
  const uint32_t tmem_base = *tmemptr;

  const uint32_t t_begin = cta_first_tile(c, G, T), t_end = cta_first_tile(c + 1, G, T);
  const EpiParams ep{pr.x_scale, reinterpret_cast<const __half *>(cv.base + cv.off_scales), cv.w_scale, pr.y, pr.ldy,
                     pr.partials, pr.counters, P.epoch, pr.m, mpad};

  // Warp roles: decoders 0..D-1, epilogue D..D+3 (TMEM lane quadrant = warp % 4), MMA issuer D+4.  The
  // scheduler favours high warp ids, so the MMA issuer reacts first: a finished unit is consumed and its
  // slot handed back to the decoders with the least delay.
  const int epi0 = int(P.D), mma_warp = int(P.D) + kEpiWarps;
  if (warp < epi0) {
    // ===================== decoder warps: Alg V.2 into the operand slots =====================
    const uint32_t d = uint32_t(warp);
    {
      const uint32_t PT = P.D / NW, team = d / NW, hw = d % NW;   // teams of NW warps fill one 128-row unit together
      const uint32_t ring_s = smem0 + ring_off + d * J * P.stream_bytes, tab_s = smem0 + tab_off;
      const uint32_t aux = LS ? ((lane & 1) ? uint32_t(-2) : 2u) : lanemask_lt();
      PairLut plut{0, 0, 0, 0};
      if constexpr (FMT == ANSLIN_FMT_BF16_PAIR4) {
        const uint4 c = *reinterpret_cast<const uint4 *>(cv.base + cv.off_scales);
        plut = PairLut{c.x, c.y, c.z, c.w};
      }
      constexpr uint32_t kUnitsPerSeg = LS ? seg_steps_of(FMT) / unit_steps32(FMT) : 1;
      const uint32_t *offs = reinterpret_cast<const uint32_t *>(cv.base + cv.off_offsets);
      const size_t rtb = raw_tile_bytes(32 * RB, cv.tile_k, PAYLOAD ? ANSLIN_FLAG_STATE_PAYLOAD : 0);
      const uint32_t xbytes = mpad * 32u;
      const int V = int(units) * RB;
      // Groups of this CTA are dealt to the teams round-robin over the CTA's WHOLE range (group i ->
      // team i mod PT, round i div PT).  The MMA warp consumes units segment by segment (one
      // accumulator per stripe segment); inside a segment the order is (round, unit, group).
      bool dep_waited = false;       // griddepcontrol.wait done (before the first load of X)
      uint32_t bsel = 0, bpar = 1;   // this team's next private slot (unit count mod B) and the parity its empty barrier must have passed
#pragma unroll 1
      for (uint32_t i = team; i < t_end - t_begin; i += PT) {
        const uint32_t gt = t_begin + i, stripe = gt / KT, kt = gt % KT;
        typename POL::S s[J];
        RawReader<PAYLOAD> raw[J];
        const uint32_t *sz[J];
        SmemEmit<RB, J> emit;
        stream_drain();
#pragma unroll
        for (int j = 0; j < J; ++j) {
          const uint32_t q = hw * J + j, t = gt * Q + q;
          const uint8_t *rec = cv.base + cv.off_records + size_t(offs[t]) * 16;
          if constexpr (LS) lane_open(s[j], rec, int(units / kUnitsPerSeg), lane);
          else stream_open(s[j], rec, ring_s + j * P.stream_bytes, lane);
          if (is_bf16_like(FMT)) raw[j].open(cv.base + cv.off_raw + size_t(t) * rtb, V, lane);
          emit.row0[j] = q * 32u * RB;
          sz[j] = nullptr;
        }
        // the record offsets of this warp's NEXT tiles: loaded now, used after the first unit to pull the records
        // (and the first raw vectors) into L2, so that the next tile switch waits for L2 rather than HBM
        const bool has_next = i + PT < t_end - t_begin;
        uint32_t next_off[J];
#pragma unroll
        for (int j = 0; j < J; ++j) next_off[j] = has_next ? offs[(gt + PT) * Q + hw * J + j] : 0u;
#pragma unroll 1
        for (uint32_t u = 0; u < units; ++u) {
          if (u == 1 && has_next) {
#pragma unroll
            for (int j = 0; j < J; ++j) {
              if (lane < 24) prefetch_l2(cv.base + cv.off_records + size_t(next_off[j]) * 16 + lane * 128);
              else if (is_bf16_like(FMT)) prefetch_l2(cv.base + cv.off_raw + size_t((gt + PT) * Q + hw * J + j) * rtb + (lane - 24) * 128);
            }
          }
          // team-private slots: unit n of this team lives in slot team*B + n % B (B = P.B buffers per team), so the
          // only thing a producer ever waits for is the MMA that read ITS OWN slot B units ago.
          const uint32_t slot = team * P.B + bsel;
          const uint32_t slot_a = slots_s + slot * P.slot_bytes;
          mbar_wait(empty_s + 8 * slot, bpar);
          if (++bsel == P.B) { bsel = 0; bpar ^= 1u; }
          const int k_elem = int(kt * cv.tile_k + u * unit_k_of(FMT));
          emit.slot_a = slot_a;
          if (FMT == ANSLIN_FMT_INT4_AWQ) {
#pragma unroll
            for (int j = 0; j < J; ++j)
              sz[j] = reinterpret_cast<const uint32_t *>(cv.base + cv.off_scales) + size_t(uint32_t(k_elem) / cv.group) * cv.n_out +
                      size_t(stripe) * kTileN + emit.row0[j];
          }
          if constexpr (LS) {
            if (u % kUnitsPerSeg == 0) {
              lane_open_segments<J>(s, ring_s, P.stream_bytes, int(u / kUnitsPerSeg), lane);
            }
          }
          if (!dep_waited) { grid_dep_wait(); dep_waited = true; }
          if (hw == 0 && lane == 0) {
            mbar_arrive_expect_tx(full_s + 8 * slot, xbytes);
            tma_load_2d(slot_a + kUnitBytes, &tms.m[pi], k_elem, 0, full_s + 8 * slot);
          }
          decode_unit<FMT, RB, J, PAYLOAD, POL>(s, ring_s, tab_s, lane, aux, int(u), V, raw, sz, emit, plut);
          fence_proxy_async();  // generic-proxy stores -> visible to the tensor core's async proxy
          __syncwarp();
          if (lane == 0) mbar_arrive(full_s + 8 * slot);
        }
      }
      cp_async_wait_all();
    }
  } else if (warp == mma_warp) {
    // ===================== MMA issuer: one thread drives the tensor core =====================
    const uint32_t idesc = make_idesc(TR::c, P.afmt, P.bfmt, 128, mpad);
    const uint32_t PT = P.D / NW, N = t_end - t_begin;
    // Consumption order: rounds of PT groups; inside a round, units ascending and groups ascending, with
    // up to TWO stripe segments of the round interleaved (they own different TMEM accumulators), so the
    // teams of a round never wait for one another's whole tile at a stripe boundary.  The order is fixed
    // by the shape alone: accumulation is bit-reproducible.
    uint32_t n_commit = 0, rel = 0;   // segments whose accumulator has been committed / handed to the epilogue
    auto release = [&](uint32_t upto, bool block) {   // hand finished accumulators to the epilogue, in segment order
      while (rel < upto && rel < n_commit) {
        const uint32_t bar = tfull_s + 8 * (rel & 1u), par = (rel >> 1) & 1u;
        if (block) mbar_wait(bar, par);
        else if (!__all_sync(0xffffffffu, mbar_test(bar, par))) break;
        named_bar_arrive(kBarEpiGo + int(rel & 1u), (kEpiWarps + 1) * 32);
        ++rel;
      }
    };
    const uint32_t stripe0 = t_begin / KT;
    // per-unit work of this warp is the serial bottleneck of the CTA once the decoders are fast (one unit per
    // ~0.3 us): descriptors are advanced by adds, segment bookkeeping is hoisted out of the unit loop
    const uint64_t adesc0 = make_smem_desc(slots_s, 16, 256, kLayoutSW32);
    const uint32_t desc_hi = uint32_t(adesc0 >> 32), adesc0_lo = uint32_t(adesc0), slot_units = P.slot_bytes >> 4;
    for (uint32_t rho = 0; rho * PT < N; ++rho) {
      const uint32_t ga = rho * PT, gb = min(N, ga + PT);
      for (uint32_t i0 = ga; i0 < gb;) {
        // run 1 = groups [i0, e1) of segment s1, run 2 = groups [e1, e2) of segment s1 + 1 (may be empty)
        const uint32_t s1 = (t_begin + i0) / KT - stripe0;
        const uint32_t e1 = min(gb, (stripe0 + s1 + 1) * KT - t_begin), e2 = min(gb, (stripe0 + s1 + 2) * KT - t_begin);
        for (uint32_t sg = s1; sg <= s1 + 1; ++sg) {   // segments that START in this window need a drained accumulator
          const uint32_t first_grp = sg == 0 ? 0u : (stripe0 + sg) * KT - t_begin;
          if (first_grp < i0 || first_grp >= e2) continue;
          if (sg >= 2) release(sg - 1, true);
          mbar_wait(tempty_s + 8 * (sg & 1u), ((sg >> 1) & 1u) ^ 1u);
          tc_fence_after();
        }
        const uint32_t first1 = s1 == 0 ? 0u : (stripe0 + s1) * KT - t_begin, last1 = min(N, (stripe0 + s1 + 1) * KT - t_begin) - 1;
        const uint32_t last2 = min(N, (stripe0 + s1 + 2) * KT - t_begin) - 1;   // segment s1 + 1 starts at e1 when it is in the window
        const uint32_t d1 = tmem_base + (s1 & 1u) * mpad, d2 = tmem_base + ((s1 + 1) & 1u) * mpad;
        const uint32_t tf1 = tfull_s + 8 * (s1 & 1u), tf2 = tfull_s + 8 * ((s1 + 1) & 1u);
        uint32_t n_unit = rho * units, bsel = n_unit % P.B, par = (n_unit / P.B) & 1u;
        for (uint32_t u = 0; u < units; ++u) {
          const bool lastu = u + 1 == units;
          // One unit ROW of the window at a time: lane l waits for the full barrier of group i0 + l (all of them in
          // parallel, instead of one barrier round trip per unit), then one thread issues the row's MMAs back to back.
          if (rel < n_commit) release(n_commit, false);
          const uint32_t slot0 = (i0 - ga) * P.B + bsel, nrow = e2 - i0;
          if (uint32_t(lane) < nrow) mbar_wait(full_s + 8 * (slot0 + uint32_t(lane) * P.B), par);
          __syncwarp();
          tc_fence_after();
          if (lane == 0) {
            uint32_t slot = slot0;
            for (uint32_t i = i0; i < e2; ++i, slot += P.B) {
              const bool run1 = i < e1;
              const bool last = lastu && i == (run1 ? last1 : last2);
              const uint32_t accumulate = (u == 0 && i == (run1 ? first1 : e1)) ? 0u : 1u;
              const uint32_t alo = adesc0_lo + slot * slot_units;   // start address field: (slots_s + slot * slot_bytes) >> 4
              const uint64_t ad = (uint64_t(desc_hi) << 32) | alo, bd = (uint64_t(desc_hi) << 32) | (alo + (kUnitBytes >> 4));
              umma<TR::kind>(run1 ? d1 : d2, ad, bd, idesc, accumulate);
              umma_commit(empty_s + 8 * slot);  // frees the slot when the MMA has read it
              if (last) umma_commit(run1 ? tf1 : tf2);
            }
          }
          __syncwarp();
          if (lastu) n_commit += (last1 >= i0 && last1 < e1 ? 1u : 0u) + (last2 >= e1 && last2 < e2 ? 1u : 0u);
          if (++bsel == P.B) { bsel = 0; par ^= 1u; }
        }
        i0 = e2;
      }
    }
    release(n_commit, true);
  } else if (warp < mma_warp) {
    // ===================== epilogue warps =====================
    grid_dep_wait();   // Y, the scales and the workspace belong to the stream's earlier kernels until they are done
    epilogue_run<FMT, YB>(ep, tmem_base, tfull_s, tempty_s, fin, t_begin, t_end, KT, c, G, T, warp & 3, lane);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == mma_warp) tmem_dealloc(tmem_base, P.tmem_cols);
  grid_dep_wait();   // warps that had no work of their own join the fix-up: same rule
  splitk_fixup<FMT, YB>(ep, fin, KT, c, G, T);
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
  uint32_t *partials;
  unsigned long long *counters;
  uint32_t epoch;
  uint32_t n_out, k_in, m, mpad, S /*stages*/, stage_bytes, tmem_cols, KB /*k blocks of 128 B*/;
  uint32_t afmt, bfmt;
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
  FinSeg *fin = reinterpret_cast<FinSeg *>(smem + bar_off + 16 * kMaxSlots + 48);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t G = gridDim.x, KT = p.KB, T = (p.n_out / kTileN) * KT;
  grid_dep_launch_dependents();   // programmatic dependent launch: the next kernel's prologue may overlap this one's tail
  if (threadIdx.x == 0) {
    for (uint32_t i = 0; i < p.S; ++i) { mbar_init(full_s + 8 * i, 1); mbar_init(empty_s + 8 * i, 1); }
    for (uint32_t i = 0; i < 2; ++i) { mbar_init(tfull_s + 8 * i, 1); mbar_init(tempty_s + 8 * i, kEpiWarps); fin[i].valid = 0; }
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc(tmemptr_s, p.tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmemptr;
  const uint32_t t_begin = cta_first_tile(blockIdx.x, G, T), t_end = cta_first_tile(blockIdx.x + 1, G, T);
  const EpiParams ep{p.x_scale, reinterpret_cast<const __half *>(p.w_scale_h), p.w_scale, p.y, p.ldy, p.partials, p.counters, p.epoch, p.m, p.mpad};

  if (warp == 5) {
    if (lane == 0) {
      uint32_t seq = 0;
      grid_dep_wait();   // W and X belong to the stream's earlier kernels until they are done; every store of this CTA follows a load
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
    const uint32_t idesc = make_idesc(TR::c, p.afmt, p.bfmt, 128, p.mpad);
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
      mbar_wait(tfull_s + 8 * ab, (si >> 1) & 1u);
      named_bar_arrive(kBarEpiGo + int(si & 1u), (kEpiWarps + 1) * 32);
      t += nt;
    }
    (void)UK;
  } else {
    epilogue_run<FMT>(ep, tmem_base, tfull_s, tempty_s, fin, t_begin, t_end, KT, blockIdx.x, G, T, warp, lane);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, p.tmem_cols);
  splitk_fixup<FMT>(ep, fin, KT, blockIdx.x, G, T);
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
// The encoded map is a function of these arguments only (it holds the address, not a device handle), and encoding costs a
// driver call: the last few maps of a thread are kept, so that a serving loop that calls with the same (pointer, m, ld)
// step after step encodes each map once.
bool make_map_2d(CUtensorMap *map, const void *ptr, int ebytes, uint64_t cols, uint64_t rows, uint64_t ld, uint32_t box_cols,
                 uint32_t box_rows, CUtensorMapSwizzle swz) {
  struct Entry { const void *ptr; uint64_t cols, rows, ld; uint32_t box_cols, box_rows; int ebytes, swz; bool valid; CUtensorMap map; };
  constexpr int kEntries = 32;
  static thread_local Entry cache[kEntries] = {};
  static thread_local int next = 0;
  for (int i = 0; i < kEntries; ++i) {
    const Entry &e = cache[i];
    if (e.valid && e.ptr == ptr && e.cols == cols && e.rows == rows && e.ld == ld && e.box_cols == box_cols && e.box_rows == box_rows &&
        e.ebytes == ebytes && e.swz == int(swz)) {
      *map = e.map;
      return true;
    }
  }
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows}, strides[1] = {ld * uint64_t(ebytes)};
  cuuint32_t box[2] = {box_cols, box_rows}, estr[2] = {1, 1};
  CUtensorMapDataType dt = ebytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_UINT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8;
  if (fn(map, dt, 2, const_cast<void *>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
         CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
    return false;
  Entry &e = cache[next];
  next = (next + 1) % kEntries;
  e.ptr = ptr; e.cols = cols; e.rows = rows; e.ld = ld; e.box_cols = box_cols; e.box_rows = box_rows; e.ebytes = ebytes; e.swz = int(swz);
  e.map = *map;
  e.valid = true;
  return true;
}

// Per-device state (SM count, "shared-memory limit raised" marks of the kernel instantiations) is indexed by the current device.
constexpr int kMaxDevices = 64;
int device_index() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) return 0;
  return dev % kMaxDevices;
}
int num_sms() {
  static std::atomic<int> n[kMaxDevices];   // 0 = not asked yet
  const int dev = device_index();
  int v = n[dev].load(std::memory_order_relaxed);
  if (v == 0) {
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    n[dev].store(v, std::memory_order_relaxed);
  }
  return v;
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

// Launch ids for the split-K counters: unique within the process and unlikely to equal whatever bytes an earlier
// owner of the workspace left behind (seeded from the clock), so the workspace never has to be cleared.
uint32_t next_epoch() {
  static std::atomic<uint32_t> e{uint32_t(std::chrono::steady_clock::now().time_since_epoch().count()) | 1u};
  uint32_t v = e.fetch_add(1, std::memory_order_relaxed);
  if (v == 0) v = e.fetch_add(1, std::memory_order_relaxed);   // 0 means "flag cleared"
  return v;
}

// bytes of a problem's split-K flag area: the shared-memory design keeps two u32 flags per CTA and a u64 counter per stripe,
// the tensor-memory design one u32 flag per (partial slot of a team, reader) = kTmFlagSlots x pairs per stripe
size_t flag_bytes(const Header &h) {
  const size_t stripes = h.n_out / kTileN, pk = h.k_in / h.tile_k;   // items per stripe: k-tile pairs, or single k-tiles (J = 1)
  return align16(std::max(stripes * 8 + 256 + 8 * 160 * kMaxTeams, kTmFlagSlots * pk * 4));
}
struct Workspace { size_t counters_off, partials_off, total; };
Workspace workspace_layout(uint32_t kb, uint32_t grid, uint32_t mpad) {   // kb: k-blocks per stripe
  Workspace w;
  w.counters_off = 0;
  w.partials_off = align16(size_t(grid) * 2 * kb * 4 + 256);   // the dense comparator's flag area: one word per (partial slot, reader)
  w.total = w.partials_off + size_t(grid) * 2 * mpad * kTileN * 4;
  return w;
}

bool x_dtype_ok(uint32_t fmt, uint32_t dt) {
  return (is_bf16_like(fmt) && dt == ANSLIN_DT_BF16) || (fmt == ANSLIN_FMT_INT4_AWQ && dt == ANSLIN_DT_F16) ||
         (fmt == ANSLIN_FMT_INT8 && dt == ANSLIN_DT_I8) || (is_fp8_path(fmt) && (dt == ANSLIN_DT_FP8_E4M3 || dt == ANSLIN_DT_FP8_E5M2));
}
// tcgen05 instruction-descriptor format code of the weight operand (a) / of X (b)
uint32_t afmt_of(uint32_t fmt) { return is_bf16_like(fmt) || fmt == ANSLIN_FMT_INT8 || fmt == ANSLIN_FMT_FP8_E5M2 ? 1u : 0u; }
uint32_t bfmt_of(uint32_t fmt, uint32_t dt) { return is_fp8_path(fmt) ? (dt == ANSLIN_DT_FP8_E5M2 ? 1u : 0u) : afmt_of(fmt); }

int sm_budget() { return std::max(1, num_sms()); }

template <uint32_t FMT, int RB, bool PAYLOAD, bool LS, bool YB>
int launch_fused_y(const TensorMaps &tms, const FusedParams &p, uint32_t grid, size_t smem, cudaStream_t st) {
  auto kern = fused_gemm_kernel<FMT, RB, (RB == 1 ? kJ32 : 1), PAYLOAD, LS, YB>;
  static thread_local size_t smem_set_dev[kMaxDevices] = {};   // per instantiation and device: raise the dynamic shared memory limit once
  size_t &smem_set = smem_set_dev[device_index()];
  if (smem > smem_set) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kSmemMax)) != cudaSuccess) return ANSLIN_ERR_CUDA;
    smem_set = kSmemMax;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(32 * (kFirstDecWarp + p.D));
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // lets the kernel's prologue overlap its predecessor's tail
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, kern, tms, p) != cudaSuccess) return ANSLIN_ERR_CUDA;
  return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}

// Teams per CTA of the TMEM design (fused_tmem.cuh) for the largest padded batch of a launch and the staged segment size:
// bounded by tensor memory (mpad accumulator + 16 operand columns per team) and by shared memory; 0 = does not fit.
uint32_t tmem_teams(uint32_t mpad_max, uint32_t stream_bytes, uint32_t fmt, uint32_t *xdepth = nullptr, uint32_t xslices = 2) {
  uint32_t T = std::min<uint32_t>(kMaxTeams, 512u / (mpad_max + kASlotCols));
  for (; T > 0; --T)   // as many teams as tensor memory allows, with a 3-deep X ring if shared memory has room for it, else 2-deep
    for (uint32_t d = kXDepth; d >= 2; --d)
      if (tmem_smem_bytes(T, mpad_max, stream_bytes, fmt, d, xslices) <= kSmemMax) {
        if (xdepth) *xdepth = d;
        return T;
      }
  if (xdepth) *xdepth = kXDepth;
  return 0;
}
bool tmem_eligible(const Header &h) {
  return (h.flags & ANSLIN_FLAG_LANE_STREAMS) && h.tile_n == 32 && h.format != ANSLIN_FMT_BF16_PAIR4 && h.tile_k / unit_k_of(h.format) >= 2 && (h.tile_k / unit_k_of(h.format)) % 2 == 0 &&   // units come in pairs
        
         uint64_t(h.n_out / kTileN) * (h.k_in / h.tile_k) < (1u << 22);   // 32-bit split arithmetic in TeamMap
}

template <uint32_t FMT, bool PAYLOAD, bool YB, int J = 2>
int launch_tmem_y(const TensorMaps &tms, const TmemParams &p, uint32_t grid, size_t smem, cudaStream_t st) {
  auto kern = fused_tmem_kernel<FMT, PAYLOAD, YB, J>;
  static thread_local size_t smem_set_dev[kMaxDevices] = {};
  size_t &smem_set = smem_set_dev[device_index()];
  if (smem > smem_set) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kSmemMax)) != cudaSuccess) return ANSLIN_ERR_CUDA;
    smem_set = kSmemMax;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(32 * (kTeamWarps + 1) * p.T);   // T teams of four decoder warps + one issuer warp per team
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // the prologue overlaps the predecessor's tail
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, kern, tms, p) != cudaSuccess) return ANSLIN_ERR_CUDA;
  return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}
template <uint32_t FMT, bool PAYLOAD>
int launch_tmem(bool ybf, const TensorMaps &tms, const TmemParams &p, uint32_t grid, size_t smem, cudaStream_t st) {
  return ybf ? launch_tmem_y<FMT, PAYLOAD, true>(tms, p, grid, smem, st) : launch_tmem_y<FMT, PAYLOAD, false>(tms, p, grid, smem, st);
}
// one k-tile per work item (fused_tmem_kernel's J = 1): bf16 and int8 only
template <uint32_t FMT, bool PAYLOAD>
int launch_tmem_single(bool ybf, const TensorMaps &tms, const TmemParams &p, uint32_t grid, size_t smem, cudaStream_t st) {
  return ybf ? launch_tmem_y<FMT, PAYLOAD, true, 1>(tms, p, grid, smem, st) : launch_tmem_y<FMT, PAYLOAD, false, 1>(tms, p, grid, smem, st);
}

// One launch over n <= kMaxProblems independent GEMMs that share format and tile geometry.
// CTAs of a persistent launch, shared out between its problems in proportion to their sizes: each problem at least one CTA
// and at most `cap[i]`, never more than S in total when n <= S.
void share_ctas(int n, const uint64_t *work, const uint32_t *cap, uint32_t S, uint32_t *ncta) {
  uint64_t work_sum = 0;
  for (int i = 0; i < n; ++i) work_sum += work[i];
  uint32_t used = 0;
  for (int i = 0; i < n; ++i) {
    ncta[i] = uint32_t(std::min<uint64_t>(cap[i], std::max<uint64_t>(1, uint64_t(S) * work[i] / work_sum)));
    used += ncta[i];
  }
  while (used > S) {   // the one-CTA minimum of tiny problems: take CTAs back from the problem with the least work per CTA
    int worst = -1;
    for (int i = 0; i < n; ++i)
      if (ncta[i] > 1 && (worst < 0 || work[i] * ncta[worst] < work[worst] * ncta[i])) worst = i;
    if (worst < 0) break;
    --ncta[worst]; --used;
  }
  for (bool grown = true; used < S && grown;) {  // hand out what rounding left over, largest work per CTA first
    grown = false;
    int best = -1;
    for (int i = 0; i < n; ++i) {
      if (ncta[i] >= cap[i]) continue;
      if (best < 0 || work[i] * ncta[best] > work[best] * ncta[i]) best = i;
    }
    if (best >= 0) { ++ncta[best]; ++used; grown = true; }
  }
}

int gemm_launch(int n, const anslin_weight *const *ws, const void *const *xs, uint32_t x_dtype, const int64_t *ldx, const int32_t *ms,
                const void *const *x_scales, void *const *ys, const int64_t *ldy, void *workspace_dev, size_t workspace_bytes,
                cudaStream_t st, uint32_t y_dtype = ANSLIN_DT_F32) {
  if (n < 1 || n > kMaxProblems || !workspace_dev || (reinterpret_cast<uintptr_t>(workspace_dev) & 15)) return ANSLIN_ERR_INVALID_ARG;
  if (y_dtype != ANSLIN_DT_F32 && y_dtype != ANSLIN_DT_BF16) return ANSLIN_ERR_UNSUPPORTED;
  if (num_sms() <= 0) return ANSLIN_ERR_CUDA;
  const Header &h0 = ws[0]->h;
  const bool scaled = h0.format == ANSLIN_FMT_INT8 || is_fp8_path(h0.format);
  const int xb = (is_bf16_like(h0.format) || h0.format == ANSLIN_FMT_INT4_AWQ) ? 2 : 1;
  if (!x_dtype_ok(h0.format, x_dtype)) return ANSLIN_ERR_INVALID_ARG;
  uint32_t mpad_max = 16;
  uint64_t work[kMaxProblems];
  for (int i = 0; i < n; ++i) {
    const anslin_weight *w = ws[i];
    if (!w || !w->dev || !xs[i] || !ys[i]) return ANSLIN_ERR_INVALID_ARG;
    if (ms[i] < 1 || ms[i] > 256) return ANSLIN_ERR_UNSUPPORTED;
    const Header &h = w->h;
    if (h.format != h0.format || h.tile_n != h0.tile_n || h.flags != h0.flags) return ANSLIN_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(xs[i]) | reinterpret_cast<uintptr_t>(ys[i])) & 15) return ANSLIN_ERR_INVALID_ARG;
    if (scaled && !x_scales[i]) return ANSLIN_ERR_INVALID_ARG;
    if (ldx[i] < int64_t(h.k_in) || (ldx[i] * xb) % 16 || ldy[i] < int64_t(h.n_out)) return ANSLIN_ERR_INVALID_ARG;
    mpad_max = std::max(mpad_max, mpad_of(ms[i]));
    work[i] = uint64_t(h.n_out) * h.k_in;
  }
  const int RB = int(h0.tile_n) / 32, J = RB == 1 ? kJ32 : 1, NW = 4 / (RB * J);
  const bool ls = h0.flags & ANSLIN_FLAG_LANE_STREAMS;
  if (ls && RB != 1) return ANSLIN_ERR_CORRUPT;
  uint32_t stream_bytes = kStreamSmem;
  bool tmem_ok = true;
  if (ls) {
    stream_bytes = 32;
    for (int i = 0; i < n; ++i) {
      stream_bytes = std::max<uint32_t>(stream_bytes, uint32_t(align16(ws[i]->h.max_seg_bytes)));
      tmem_ok = tmem_ok && tmem_eligible(ws[i]->h);
    }
  }
  // which design: decoded operand through tensor memory (fused_tmem.cuh) or through shared-memory operand slots
  uint32_t xdepth = kXDepth, xdepth1 = kXDepth;
  uint32_t T = (ls && tmem_ok) ? tmem_teams(mpad_max, stream_bytes, h0.format, &xdepth) : 0u;
  const uint32_t T1 = (ls && tmem_ok) ? tmem_teams(mpad_max, stream_bytes, h0.format, &xdepth1, 1) : 0u;   // with one X slice per ring slot (J = 1)
  // The tensor-memory design works on pairs of k-tiles of one stripe.  A launch with fewer pairs than 0.6 x teams (few, long
  // tiles: e.g. 32 x 1024 int8 tiles of a 13824 x 5120 matrix) is bound by the sequential length of a tile pair; the
  // shared-memory design splits such a launch by single k-tiles and finishes sooner.
  uint64_t pairs = 0;
  for (int i = 0; i < n; ++i) pairs += uint64_t(ws[i]->h.n_out / kTileN) * ((ws[i]->h.k_in / ws[i]->h.tile_k + 1) / 2);
  const bool long_tiles = h0.tile_k / unit_k_of(h0.format) >= 32;
  // ... unless no team gets more than one k-tile: then the tensor-memory kernel runs with ONE tile per work item and one chain
  // per warp (J = 1), and the launch lasts one tile at a chain's latency instead of one pair at two interleaved chains'
  uint64_t tiles_total = 0;
  for (int i = 0; i < n; ++i) tiles_total += uint64_t(ws[i]->h.n_out / kTileN) * (ws[i]->h.k_in / ws[i]->h.tile_k);
  const bool single = T1 >= 2 && (h0.format == ANSLIN_FMT_BF16 || h0.format == ANSLIN_FMT_INT8) && tiles_total <= uint64_t(sm_budget()) * T1;
  if (single) { T = T1; xdepth = xdepth1; }
  const bool use_tmem = T >= 2 && (single || !(long_tiles && pairs * 10 < uint64_t(sm_budget()) * T * 6));
  // CTAs: one per SM in total, shared out in proportion to the problems' sizes
  const uint32_t S = uint32_t(sm_budget());
  uint32_t ncta[kMaxProblems], cap[kMaxProblems];
  for (int i = 0; i < n; ++i) cap[i] = (ws[i]->h.n_out / kTileN) * (ws[i]->h.k_in / ws[i]->h.tile_k);
  share_ctas(n, work, cap, S, ncta);
  // workspace: flags of all problems, then the split-K partials (two per CTA, or two per team)
  const uint32_t teams = use_tmem ? T : 1u;
  size_t off = 0;
  uint8_t *wsb = static_cast<uint8_t *>(workspace_dev);
  size_t counters_bytes = 0;
  for (int i = 0; i < n; ++i) counters_bytes += flag_bytes(ws[i]->h);
  size_t part_off = counters_bytes;
  uint32_t cta0 = 0;
  Problem prob[kMaxProblems];
  TensorMaps tms;
  for (int i = 0; i < n; ++i) {
    const Header &h = ws[i]->h;
    Problem &q = prob[i];
    q.cv = view_of(ws[i]);
    q.x_scale = static_cast<const float *>(x_scales ? x_scales[i] : nullptr);
    q.y = static_cast<float *>(ys[i]);
    q.ldy = ldy[i];
    q.m = uint32_t(ms[i]);
    q.mpad = mpad_of(ms[i]);
    q.cta0 = cta0;
    q.ncta = ncta[i];
    cta0 += ncta[i];
    q.counters = reinterpret_cast<unsigned long long *>(wsb + off);
    off += flag_bytes(h);
    q.partials = reinterpret_cast<uint32_t *>(wsb + part_off);
    part_off += size_t(ncta[i]) * teams * 2 * q.mpad * kTileN * 4;
    const uint32_t uk = unit_k_of(h.format);
    if (!make_map_2d(&tms.m[i], xs[i], xb, h.k_in, uint64_t(ms[i]), uint64_t(ldx[i]), uk, q.mpad, CU_TENSOR_MAP_SWIZZLE_32B))
      return ANSLIN_ERR_CUDA;
  }
  if (workspace_bytes < part_off) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  const uint32_t grid = cta0;
  const bool ybf = y_dtype == ANSLIN_DT_BF16;
  const bool pay = h0.flags & ANSLIN_FLAG_STATE_PAYLOAD;
  if (use_tmem) {
    TmemParams p;
    memset(&p, 0, sizeof(p));
    memcpy(p.prob, prob, sizeof(Problem) * size_t(n));
    p.nprob = uint32_t(n);
    p.T = T;
    p.epoch = next_epoch();
    p.stream_bytes = stream_bytes;
    p.xslice_bytes = mpad_max * 32u;
    p.tmem_stride = mpad_max + kASlotCols;
    p.afmt = afmt_of(h0.format); p.bfmt = bfmt_of(h0.format, x_dtype);
    p.xdepth = xdepth;
    const size_t smem = tmem_smem_bytes(T, mpad_max, stream_bytes, h0.format, xdepth, single ? 1u : 2u);
    switch (h0.format) {
      case ANSLIN_FMT_BF16:
        if (single) return pay ? launch_tmem_single<ANSLIN_FMT_BF16, true>(ybf, tms, p, grid, smem, st) : launch_tmem_single<ANSLIN_FMT_BF16, false>(ybf, tms, p, grid, smem, st);
        return pay ? launch_tmem<ANSLIN_FMT_BF16, true>(ybf, tms, p, grid, smem, st) : launch_tmem<ANSLIN_FMT_BF16, false>(ybf, tms, p, grid, smem, st);
      case ANSLIN_FMT_FP8_E4M3:
      case ANSLIN_FMT_FP8_E5M2: return launch_tmem<ANSLIN_FMT_FP8_E4M3, false>(ybf, tms, p, grid, smem, st);
      case ANSLIN_FMT_INT8: return single ? launch_tmem_single<ANSLIN_FMT_INT8, false>(ybf, tms, p, grid, smem, st) : launch_tmem<ANSLIN_FMT_INT8, false>(ybf, tms, p, grid, smem, st);
      case ANSLIN_FMT_INT4_AWQ: return launch_tmem<ANSLIN_FMT_INT4_AWQ, false>(ybf, tms, p, grid, smem, st);
      case ANSLIN_FMT_FP4_E2M1: return launch_tmem<ANSLIN_FMT_FP4_E2M1, false>(ybf, tms, p, grid, smem, st);
    }
    return ANSLIN_ERR_UNSUPPORTED;
  }
  FusedParams p;
  memset(&p, 0, sizeof(p));
  memcpy(p.prob, prob, sizeof(Problem) * size_t(n));
  p.nprob = uint32_t(n);
  p.slot_bytes = kUnitBytes + mpad_max * 32u;
  p.tmem_cols = tmem_cols_of(mpad_max);
  // shared memory: U operand slots, D*J stream rings, slot table, barriers
  const size_t fixed = 2048 /*align slack*/ + 16384 + 1056 + 16 * kMaxSlots + 96;
  p.stream_bytes = stream_bytes;
  uint32_t D = kMaxDecWarps, U = 0;
  D -= D % NW;
  uint32_t Bslots = 0;
  for (; D >= uint32_t(NW); D -= NW) {   // most decoder warps that still leave every team two private operand slots
    const size_t rings = size_t(D) * J * stream_bytes;
    if (kSmemMax < fixed + rings) continue;
    const uint32_t PT = D / NW;
    Bslots = uint32_t(std::min<size_t>((kSmemMax - fixed - rings) / p.slot_bytes, kMaxSlots) / PT);
    if (Bslots >= 2) break;
  }
  if (D < uint32_t(NW) || Bslots < 2) return ANSLIN_ERR_UNSUPPORTED;
  Bslots = std::min(Bslots, 6u);
  U = (D / NW) * Bslots;
  p.D = D;
  p.U = U;
  p.B = Bslots;
  const size_t smem = fixed + size_t(D) * J * stream_bytes + size_t(U) * p.slot_bytes;
  p.epoch = next_epoch();
  p.afmt = afmt_of(h0.format); p.bfmt = bfmt_of(h0.format, x_dtype);
#define launch_fused(...) (ybf ? launch_fused_y<__VA_ARGS__, true>(tms, p, grid, smem, st) : launch_fused_y<__VA_ARGS__, false>(tms, p, grid, smem, st))
#define ANSLIN_LAUNCH(F, PAY)                                                                                   \
  (RB == 1 ? (ls ? launch_fused(F, 1, PAY, true) : launch_fused(F, 1, PAY, false)) \
           : launch_fused(F, 4, PAY, false))
  switch (h0.format) {
    case ANSLIN_FMT_BF16: return pay ? ANSLIN_LAUNCH(ANSLIN_FMT_BF16, true) : ANSLIN_LAUNCH(ANSLIN_FMT_BF16, false);
    case ANSLIN_FMT_BF16_PAIR4:   // lane streams on 32-row tiles only (anslin_open checked)
      if (RB != 1 || !ls) return ANSLIN_ERR_CORRUPT;
      return pay ? launch_fused(ANSLIN_FMT_BF16_PAIR4, 1, true, true) : launch_fused(ANSLIN_FMT_BF16_PAIR4, 1, false, true);
    case ANSLIN_FMT_FP8_E4M3:
    case ANSLIN_FMT_FP8_E5M2: return ANSLIN_LAUNCH(ANSLIN_FMT_FP8_E4M3, false);   // same bytes, another descriptor code
    case ANSLIN_FMT_INT8: return ANSLIN_LAUNCH(ANSLIN_FMT_INT8, false);
    case ANSLIN_FMT_INT4_AWQ: return ANSLIN_LAUNCH(ANSLIN_FMT_INT4_AWQ, false);
    case ANSLIN_FMT_FP4_E2M1: return ANSLIN_LAUNCH(ANSLIN_FMT_FP4_E2M1, false);
  }
#undef ANSLIN_LAUNCH
#undef launch_fused
  return ANSLIN_ERR_UNSUPPORTED;
}

size_t multi_workspace_bytes(const anslin_weight *const *ws, int n, int32_t m_max) {
  if (!ws || n < 1 || m_max < 1 || m_max > 256) return 0;
  size_t counters = 0;
  uint32_t stream_bytes = 32;
  bool tmem_ok = true;
  for (int i = 0; i < n; ++i) {
    if (!ws[i]) return 0;
    counters += flag_bytes(ws[i]->h);
    stream_bytes = std::max<uint32_t>(stream_bytes, uint32_t(align16(ws[i]->h.max_seg_bytes)));
    tmem_ok = tmem_ok && tmem_eligible(ws[i]->h);
  }
  // all problems of a launch share one CTA per SM, so their partials never exceed one problem's worst case: two partials
  // per CTA, or per team of the tensor-memory design (a smaller batch may run with more teams: take the largest
  // teams x mpad product up to m_max)
  size_t rows = mpad_of(m_max);
  if (tmem_ok)
    for (uint32_t mp = 16; mp <= mpad_of(m_max); mp += 16) {
      const uint32_t T = std::max(tmem_teams(mp, stream_bytes, ws[0]->h.format), tmem_teams(mp, stream_bytes, ws[0]->h.format, nullptr, 1));
      if (T >= 2) rows = std::max(rows, size_t(T) * mp);
    }
  const size_t per_launch = size_t(std::max(sm_budget(), 148)) * 2 * rows * kTileN * 4;
  return counters + per_launch;
}

template <uint32_t FMT, int RB, bool PAYLOAD, bool LS>
int launch_decode_t(const ContainerView &cv, void *out, cudaStream_t st) {
  constexpr int J = RB == 1 ? kJ32 : 1;
  const uint32_t jobs = cv.n_tiles / J;
  auto kern = decode_kernel<FMT, RB, J, PAYLOAD, LS>;
  const uint32_t stream_bytes = LS ? uint32_t(align16(std::max<uint32_t>(cv.max_seg_bytes, 32))) : kStreamSmem;
  // + 16: a lane-stream's look-ahead word load may touch the two bytes after the last stream buffer
  const size_t smem = 4 * kM + 1056 + size_t(kDecWarps) * J * (stream_bytes + GlobalEmit<FMT, RB, J>::kStageBytes) + 16;
  if (smem > kSmemMax) return ANSLIN_ERR_UNSUPPORTED;
  struct DevState { size_t smem_set, smem_occ; int occ; };
  static thread_local DevState dev_state[kMaxDevices] = {};   // per instantiation and device
  DevState &ds = dev_state[device_index()];
  size_t &smem_set = ds.smem_set, &smem_occ = ds.smem_occ;
  int &occ = ds.occ;
  if (smem > smem_set) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess) return ANSLIN_ERR_CUDA;
    smem_set = smem;
  }
  if (smem != smem_occ) {
    // one resident wave: the grid is exactly what fits on the SMs at this shared-memory size, warps loop over jobs
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kDecWarps * 32, smem) != cudaSuccess || occ < 1) return ANSLIN_ERR_CUDA;
    smem_occ = smem;
  }
  uint32_t per_sm = uint32_t(occ);
  const uint32_t ctas = std::min<uint32_t>((jobs + kDecWarps - 1) / kDecWarps, uint32_t(sm_budget()) * per_sm);
  kern<<<ctas, kDecWarps * 32, smem, st>>>(cv, static_cast<uint8_t *>(out), stream_bytes);
  return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}
// decode_lanes_kernel (decode_lanes.cuh) where the container allows it: lane streams, 32-row tiles, a unit of 32 bytes of W per
// row, an even number of units per tile, staged segments small enough for 16 decoder warps.
template <uint32_t FMT, bool PAYLOAD>
int launch_decode_lanes(const ContainerView &cv, void *out, cudaStream_t st, bool *launched) {
  *launched = false;
  if constexpr (decode_lanes_format(FMT)) {
    if (!(cv.flags & ANSLIN_FLAG_LANE_STREAMS) || cv.tile_n != 32 || cv.units < 2 || cv.units % 2 || cv.n_tiles < 2) return ANSLIN_OK;
    const uint32_t stream_bytes = uint32_t(align16(std::max<uint32_t>(cv.max_seg_bytes, 32)));
    // all 16 decoder warps or the old kernel: with fewer (int8: 4.7 KiB staged per segment) decode_kernel's 2 x 8 warps per SM win
    const uint32_t warps = kLaneDecWarps;
    if (decode_lanes_smem(FMT, warps, stream_bytes) > kSmemMax) return ANSLIN_OK;
    const size_t row_bytes = row_bytes_of(FMT, cv.k_in);
    CUtensorMap tmo;
    if (!make_map_2d(&tmo, out, 1, row_bytes, cv.n_out, row_bytes, decode_lanes_box_row(FMT), 32, CU_TENSOR_MAP_SWIZZLE_NONE)) return ANSLIN_ERR_CUDA;
    auto kern = decode_lanes_kernel<FMT, PAYLOAD>;
    static thread_local size_t smem_set_dev[kMaxDevices] = {};
    size_t &smem_set = smem_set_dev[device_index()];
    if (smem_set == 0) {
      if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kSmemMax)) != cudaSuccess) return ANSLIN_ERR_CUDA;
      smem_set = kSmemMax;
    }
    const uint32_t jobs = cv.n_tiles / 2;
    const uint32_t grid = std::min<uint32_t>(uint32_t(sm_budget()), jobs);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(warps * 32);
    cfg.dynamicSmemBytes = decode_lanes_smem(FMT, warps, stream_bytes);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // launch latency and CTA set-up overlap the predecessor's tail
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    *launched = true;
    if (cudaLaunchKernelEx(&cfg, kern, tmo, cv, stream_bytes) != cudaSuccess) return ANSLIN_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
  }
  return ANSLIN_OK;
}

template <uint32_t FMT, bool PAYLOAD>
int launch_decode(const ContainerView &cv, void *out, cudaStream_t st) {
  bool launched = false;
  const int rc = launch_decode_lanes<FMT, PAYLOAD>(cv, out, st, &launched);
  if (rc != ANSLIN_OK || launched) return rc;
  if (cv.flags & ANSLIN_FLAG_LANE_STREAMS) return cv.tile_n == 32 ? launch_decode_t<FMT, 1, PAYLOAD, true>(cv, out, st) : int(ANSLIN_ERR_CORRUPT);
  return cv.tile_n == 32 ? launch_decode_t<FMT, 1, PAYLOAD, false>(cv, out, st) : launch_decode_t<FMT, 4, PAYLOAD, false>(cv, out, st);
}

template <uint32_t FMT>
int launch_dense(const CUtensorMap &tmw, const CUtensorMap &tmx, DenseParams &p, uint32_t grid, size_t smem, cudaStream_t st) {
  auto kern = dense_gemm_kernel<FMT>;
  static thread_local size_t smem_set_dev[kMaxDevices] = {};
  size_t &smem_set = smem_set_dev[device_index()];
  if (smem > smem_set) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kSmemMax)) != cudaSuccess) return ANSLIN_ERR_CUDA;
    smem_set = kSmemMax;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(kDenseThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // the prologue overlaps the predecessor's tail
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, kern, tmw, tmx, p) != cudaSuccess) return ANSLIN_ERR_CUDA;
  return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}

}  // namespace

extern "C" {

#ifdef ANSLIN_TRACE
int anslin_debug_trace(void *host_out, size_t bytes) {
  return cudaMemcpyFromSymbol(host_out, g_trace, std::min(bytes, sizeof(g_trace))) == cudaSuccess ? 0 : 5;
}
int anslin_debug_prof(void *host_out, size_t bytes) {
  return cudaMemcpyFromSymbol(host_out, g_prof, std::min(bytes, sizeof(g_prof))) == cudaSuccess ? 0 : 5;
}
#endif

// Kernels a GEMM call enqueues, from its shape alone: its problems are cut into blocks of <= 256 batch rows and every
// launch takes up to eight blocks.
int anslin_gemm_launches(int64_t row_blocks) { return row_blocks < 1 ? 0 : int((row_blocks + kMaxProblems - 1) / kMaxProblems); }

int anslin_decode(const anslin_weight *w, void *w_out_dev, size_t capacity, void *stream) {
  if (!w || !w->dev || !w_out_dev) return ANSLIN_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(w_out_dev) & 15) return ANSLIN_ERR_INVALID_ARG;
  const Header &h = w->h;
  const size_t need = size_t(h.n_out) * row_bytes_of(h.format, h.k_in);
  if (capacity < need) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  if (num_sms() <= 0) return ANSLIN_ERR_CUDA;
  const ContainerView cv = view_of(w);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  switch (h.format) {
    case ANSLIN_FMT_BF16:
      return (h.flags & ANSLIN_FLAG_STATE_PAYLOAD) ? launch_decode<ANSLIN_FMT_BF16, true>(cv, w_out_dev, st)
                                                    : launch_decode<ANSLIN_FMT_BF16, false>(cv, w_out_dev, st);
    case ANSLIN_FMT_BF16_PAIR4:
      if (cv.tile_n != 32 || !(cv.flags & ANSLIN_FLAG_LANE_STREAMS)) return ANSLIN_ERR_CORRUPT;
      return (h.flags & ANSLIN_FLAG_STATE_PAYLOAD) ? launch_decode_t<ANSLIN_FMT_BF16_PAIR4, 1, true, true>(cv, w_out_dev, st)
                                                    : launch_decode_t<ANSLIN_FMT_BF16_PAIR4, 1, false, true>(cv, w_out_dev, st);
    case ANSLIN_FMT_FP8_E4M3:
    case ANSLIN_FMT_FP8_E5M2: return launch_decode<ANSLIN_FMT_FP8_E4M3, false>(cv, w_out_dev, st);
    case ANSLIN_FMT_INT8: return launch_decode<ANSLIN_FMT_INT8, false>(cv, w_out_dev, st);
    case ANSLIN_FMT_INT4_AWQ: return launch_decode<ANSLIN_FMT_INT4_AWQ, false>(cv, w_out_dev, st);
    case ANSLIN_FMT_FP4_E2M1: return launch_decode<ANSLIN_FMT_FP4_E2M1, false>(cv, w_out_dev, st);
  }
  return ANSLIN_ERR_UNSUPPORTED;
}

// m > 256 (S: §8(f) NEXT-1, the paper's prefill workloads P:l.392): X is cut into blocks of kMaxM rows, each block a
// problem of its own inside one persistent launch (kMaxProblems blocks per launch).  Every block decodes W again:
// correct at any m, but the decoded tile is not shared between blocks.
constexpr int32_t kMaxM = 256;

size_t anslin_gemm_workspace_bytes(const anslin_weight *w, int32_t m) {
  if (m <= kMaxM) return multi_workspace_bytes(&w, 1, m);
  const anslin_weight *ws[kMaxProblems];
  const int n = int(std::min<int64_t>(kMaxProblems, (int64_t(m) + kMaxM - 1) / kMaxM));
  for (int i = 0; i < n; ++i) ws[i] = w;
  return multi_workspace_bytes(ws, n, kMaxM);
}

size_t anslin_gemm_multi_workspace_bytes(const anslin_weight *const *weights, int32_t n, int32_t m_max) {
  return multi_workspace_bytes(weights, n, m_max);
}

int anslin_gemm(const anslin_weight *w, const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m, const void *x_scale_dev,
                void *y_dev, int64_t ldy, void *workspace_dev, size_t workspace_bytes, void *stream) {
  if (!w) return ANSLIN_ERR_INVALID_ARG;
  if (m <= kMaxM)
    return gemm_launch(1, &w, &x_dev, x_dtype, &ldx, &m, &x_scale_dev, &y_dev, &ldy, workspace_dev, workspace_bytes,
                       static_cast<cudaStream_t>(stream));
  if (!x_dev || !y_dev) return ANSLIN_ERR_INVALID_ARG;
  const int xb = (is_bf16_like(w->h.format) || w->h.format == ANSLIN_FMT_INT4_AWQ) ? 2 : 1;
  for (int32_t r0 = 0; r0 < m;) {
    const anslin_weight *ws[kMaxProblems];
    const void *xs[kMaxProblems], *xsc[kMaxProblems];
    void *ys[kMaxProblems];
    int64_t ldxs[kMaxProblems], ldys[kMaxProblems];
    int32_t ms[kMaxProblems];
    int cnt = 0;
    for (; cnt < kMaxProblems && r0 < m; ++cnt, r0 += kMaxM) {
      ws[cnt] = w;
      xs[cnt] = static_cast<const uint8_t *>(x_dev) + size_t(r0) * ldx * xb;
      xsc[cnt] = x_scale_dev ? static_cast<const float *>(x_scale_dev) + r0 : nullptr;
      ys[cnt] = static_cast<float *>(y_dev) + size_t(r0) * ldy;
      ldxs[cnt] = ldx; ldys[cnt] = ldy; ms[cnt] = std::min(kMaxM, m - r0);
    }
    const int rc = gemm_launch(cnt, ws, xs, x_dtype, ldxs, ms, xsc, ys, ldys, workspace_dev, workspace_bytes, static_cast<cudaStream_t>(stream));
    if (rc != ANSLIN_OK) return rc;
  }
  return ANSLIN_OK;
}

// ---- anslin_gemm without a caller-provided workspace and without any allocation ------------------------------------------
// The split-K flags and partials live in a file-scope device array (every GPU that loads the library holds these
// ANSLIN_STATIC_WORKSPACE_BYTES until the process exits).  In host code the array's NAME is only a host-side stand-in for the
// symbol, never a device address: its address is asked for once per device with cudaGetSymbolAddress, with that device
// current, and that pointer is what the kernel is given.
static __device__ __align__(256) unsigned char g_static_workspace[ANSLIN_STATIC_WORKSPACE_BYTES];

int anslin_gemm_static(const anslin_weight *w, const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m, const void *x_scale_dev,
                       void *y_dev, int64_t ldy, void *stream) {
  if (!w) return ANSLIN_ERR_INVALID_ARG;
  if (m < 1) return ANSLIN_ERR_INVALID_ARG;
  // the same size rule as the caller of anslin_gemm follows; beyond the array: refuse before anything is enqueued
  const size_t need = anslin_gemm_workspace_bytes(w, m);
  if (need == 0) return ANSLIN_ERR_UNSUPPORTED;
  if (need > size_t(ANSLIN_STATIC_WORKSPACE_BYTES)) return ANSLIN_ERR_STATIC_LIMIT;
  constexpr int kMaxDevices = 64;
  static std::atomic<void *> ptr_of_device[kMaxDevices];   // zero-initialised; a race between two first calls stores the same value twice
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return ANSLIN_ERR_CUDA;
  void *ptr = ptr_of_device[dev].load(std::memory_order_acquire);
  if (!ptr) {
    if (cudaGetSymbolAddress(&ptr, g_static_workspace) != cudaSuccess || !ptr) return ANSLIN_ERR_CUDA;
    ptr_of_device[dev].store(ptr, std::memory_order_release);
  }
  // The array keeps whatever the last call left in it.  The kernels need the split-K flag words to start as "not stored":
  // their readers take them down and a flag holds a per-launch epoch, but this path does not lean on either: the flag
  // area (the first bytes of the workspace; the partials behind it are written before they are read) is cleared
  // on the stream ahead of the launch.  No allocation: a memset node, capturable like the launch itself.
  const size_t flags = flag_bytes(w->h) * size_t(std::max<int64_t>(1, std::min<int64_t>(kMaxProblems, (int64_t(m) + kMaxM - 1) / kMaxM)));
  if (cudaMemsetAsync(ptr, 0, std::min(flags, need), static_cast<cudaStream_t>(stream)) != cudaSuccess) return ANSLIN_ERR_CUDA;
  return anslin_gemm(w, x_dev, x_dtype, ldx, m, x_scale_dev, y_dev, ldy, ptr, size_t(ANSLIN_STATIC_WORKSPACE_BYTES), stream);
}

int anslin_gemm_multi_ex(const anslin_weight *const *weights, int32_t n, const void *const *x_dev, uint32_t x_dtype, const int64_t *ldx,
                         const int32_t *m, const void *const *x_scale_dev, void *const *y_dev, uint32_t y_dtype, const int64_t *ldy,
                         void *workspace_dev, size_t workspace_bytes, void *stream) {
  if (!weights || n < 1 || !x_dev || !ldx || !m || !y_dev || !ldy) return ANSLIN_ERR_INVALID_ARG;
  const void *no_scales[kMaxProblems] = {nullptr};
  for (int32_t i0 = 0; i0 < n; i0 += kMaxProblems) {   // more than kMaxProblems: consecutive launches on the same stream
    const int cnt = std::min<int32_t>(kMaxProblems, n - i0);
    int rc = gemm_launch(cnt, weights + i0, x_dev + i0, x_dtype, ldx + i0, m + i0, x_scale_dev ? x_scale_dev + i0 : no_scales, y_dev + i0,
                         ldy + i0, workspace_dev, workspace_bytes, static_cast<cudaStream_t>(stream), y_dtype);
    if (rc != ANSLIN_OK) return rc;
  }
  return ANSLIN_OK;
}

int anslin_gemm_multi(const anslin_weight *const *weights, int32_t n, const void *const *x_dev, uint32_t x_dtype, const int64_t *ldx,
                      const int32_t *m, const void *const *x_scale_dev, void *const *y_dev, const int64_t *ldy, void *workspace_dev,
                      size_t workspace_bytes, void *stream) {
  return anslin_gemm_multi_ex(weights, n, x_dev, x_dtype, ldx, m, x_scale_dev, y_dev, ANSLIN_DT_F32, ldy, workspace_dev, workspace_bytes, stream);
}

int anslin_gemm_grouped(const anslin_weight *const *experts, int32_t n_experts, const int32_t *rows_per_expert_host,
                        const void *x_dev, uint32_t x_dtype, int64_t ldx, const void *x_scale_dev, void *y_dev, int64_t ldy,
                        void *workspace_dev, size_t workspace_bytes, void *stream) {
  if (!experts || n_experts < 1 || !rows_per_expert_host || !x_dev || !y_dev) return ANSLIN_ERR_INVALID_ARG;
  // active experts -> problems of one persistent launch (kMaxProblems per launch)
  const anslin_weight *w[kMaxProblems];
  const void *xs[kMaxProblems], *xsc[kMaxProblems];
  void *ys[kMaxProblems];
  int64_t ldxs[kMaxProblems], ldys[kMaxProblems];
  int32_t ms[kMaxProblems];
  int cnt = 0;
  int64_t row = 0;
  auto flush = [&]() -> int {
    if (cnt == 0) return ANSLIN_OK;
    const int rc = gemm_launch(cnt, w, xs, x_dtype, ldxs, ms, xsc, ys, ldys, workspace_dev, workspace_bytes, static_cast<cudaStream_t>(stream));
    cnt = 0;
    return rc;
  };
  for (int e = 0; e < n_experts; ++e) {
    const int32_t rows = rows_per_expert_host[e];
    if (rows < 0 || !experts[e]) return ANSLIN_ERR_INVALID_ARG;
    if (rows == 0) continue;
    const Header &h = experts[e]->h;
    if (h.format != experts[0]->h.format || h.n_out != experts[0]->h.n_out || h.k_in != experts[0]->h.k_in) return ANSLIN_ERR_INVALID_ARG;
    const int xb = (is_bf16_like(h.format) || h.format == ANSLIN_FMT_INT4_AWQ) ? 2 : 1;
    for (int32_t r0 = 0; r0 < rows; r0 += kMaxM) {   // an expert with more than kMaxM rows is several problems (see anslin_gemm)
      if (cnt == kMaxProblems) {
        const int rc = flush();
        if (rc != ANSLIN_OK) return rc;
      }
      w[cnt] = experts[e];
      xs[cnt] = static_cast<const uint8_t *>(x_dev) + size_t(row + r0) * ldx * xb;   // row offsets keep 16-byte alignment only if the pitch does
      xsc[cnt] = x_scale_dev ? static_cast<const float *>(x_scale_dev) + row + r0 : nullptr;
      ys[cnt] = static_cast<float *>(y_dev) + size_t(row + r0) * ldy;
      ldxs[cnt] = ldx; ldys[cnt] = ldy; ms[cnt] = std::min(kMaxM, rows - r0);
      ++cnt;
    }
    row += rows;
  }
  return flush();
}

size_t anslin_dense_workspace_bytes(uint32_t n_out, uint32_t k_in, int32_t m) {
  if (m < 1 || m > 256 || n_out % kTileN) return 0;
  return workspace_layout(k_in / 64 + 1, uint32_t(std::max(num_sms(), 148)), mpad_of(m)).total;   // k-blocks of 64 (2-byte) or 128 (1-byte) elements
}

int anslin_dense_gemm(uint32_t format, const void *w_dev, uint32_t n_out, uint32_t k_in, const void *w_scale_dev, float w_scale,
                      const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m, const void *x_scale_dev, void *y_dev,
                      int64_t ldy, void *workspace_dev, size_t workspace_bytes, void *stream) {
  if (!w_dev || !x_dev || !y_dev || !workspace_dev) return ANSLIN_ERR_INVALID_ARG;
  if (format > kFormatMax || m < 1 || m > 256) return ANSLIN_ERR_UNSUPPORTED;
  // the int4 slot takes fp16 weights (what AWQ dequantises to): same MMA kind as the fused int4 path
  const uint32_t xd_need = format == ANSLIN_FMT_INT4_AWQ ? ANSLIN_DT_F16 : 0;
  if (format == ANSLIN_FMT_INT4_AWQ ? x_dtype != xd_need : !x_dtype_ok(format, x_dtype)) return ANSLIN_ERR_INVALID_ARG;
  const int xb = (is_bf16_like(format) || format == ANSLIN_FMT_INT4_AWQ) ? 2 : 1;
  const uint32_t ke = 128 / xb;
  if (n_out % kTileN || k_in % ke) return ANSLIN_ERR_UNSUPPORTED;
  if ((reinterpret_cast<uintptr_t>(w_dev) | reinterpret_cast<uintptr_t>(x_dev) | reinterpret_cast<uintptr_t>(y_dev) |
       reinterpret_cast<uintptr_t>(workspace_dev)) & 15)
    return ANSLIN_ERR_INVALID_ARG;
  const bool scaled = format == ANSLIN_FMT_INT8 || is_fp8_path(format);
  if (scaled && !x_scale_dev) return ANSLIN_ERR_INVALID_ARG;
  if (format == ANSLIN_FMT_INT8 && !w_scale_dev) return ANSLIN_ERR_INVALID_ARG;
  if (num_sms() <= 0) return ANSLIN_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  DenseParams p;
  p.w_scale_h = w_scale_dev; p.w_scale = w_scale; p.x_scale = static_cast<const float *>(x_scale_dev);
  p.y = static_cast<float *>(y_dev); p.ldy = ldy; p.n_out = n_out; p.k_in = k_in; p.m = uint32_t(m); p.mpad = mpad_of(m);
  p.KB = k_in / ke;
  p.afmt = afmt_of(format); p.bfmt = bfmt_of(format, x_dtype);
  p.stage_bytes = 16384 + p.mpad * 128u;
  p.tmem_cols = tmem_cols_of(p.mpad);
  const size_t fixed = 1024 + 16 * kMaxSlots + 96;
  p.S = uint32_t(std::min<size_t>((kSmemMax - fixed) / p.stage_bytes, 12));
  const size_t smem = fixed + size_t(p.S) * p.stage_bytes;
  const uint32_t stripes = n_out / kTileN, T = stripes * p.KB, grid = grid_of(T, 8);
  const Workspace ws = workspace_layout(p.KB, grid, p.mpad);
  if (workspace_bytes < ws.total) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  p.counters = reinterpret_cast<unsigned long long *>(static_cast<uint8_t *>(workspace_dev) + ws.counters_off);
  p.epoch = next_epoch();
  p.partials = reinterpret_cast<uint32_t *>(static_cast<uint8_t *>(workspace_dev) + ws.partials_off);
  CUtensorMap tmw, tmx;
  if (!make_map_2d(&tmw, w_dev, xb, k_in, n_out, k_in, ke, kTileN, CU_TENSOR_MAP_SWIZZLE_128B)) return ANSLIN_ERR_CUDA;
  if (!make_map_2d(&tmx, x_dev, xb, k_in, uint64_t(m), uint64_t(ldx), ke, p.mpad, CU_TENSOR_MAP_SWIZZLE_128B)) return ANSLIN_ERR_CUDA;
  switch (format) {
    case ANSLIN_FMT_BF16:
    case ANSLIN_FMT_BF16_PAIR4: return launch_dense<ANSLIN_FMT_BF16>(tmw, tmx, p, grid, smem, st);
    case ANSLIN_FMT_INT4_AWQ: return launch_dense<ANSLIN_FMT_INT4_AWQ>(tmw, tmx, p, grid, smem, st);
    case ANSLIN_FMT_FP8_E4M3:
    case ANSLIN_FMT_FP8_E5M2:
    case ANSLIN_FMT_FP4_E2M1:   // the fp4 slot takes the e4m3 bytes fp4 expands to: same MMA kind as the fused fp4 path
      return launch_dense<ANSLIN_FMT_FP8_E4M3>(tmw, tmx, p, grid, smem, st);
    case ANSLIN_FMT_INT8: return launch_dense<ANSLIN_FMT_INT8>(tmw, tmx, p, grid, smem, st);
  }
  return ANSLIN_ERR_UNSUPPORTED;
}

}  // extern "C"
