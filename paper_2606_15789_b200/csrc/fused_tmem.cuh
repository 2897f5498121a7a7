// Fused rANS-decode + tcgen05 GEMM, second design: the decoded weights reach the tensor core through TENSOR MEMORY.
// Included by kernels.cu inside its anonymous namespace (after the PTX wrappers, FmtTraits, Problem, TensorMaps).
//
// Alg V.1 (P:l.196-252) for lane-stream containers with 32-row tiles, re-cut for sm_100a:
//   * a TEAM = 4 decoder warps = one 128-row stripe; warp q of a team owns TMEM lane quadrant q, so lane l of warp q
//     IS row 32q+l of the MMA's A operand: the 16 weights (32 operand bytes) a lane decodes per unit go from its
//     registers into 8 TMEM columns with one tcgen05.st — no shared-memory operand slot, no swizzle, no proxy fence
//     ("writes the decoded value directly into the shared-memory" P:l.254 becomes "into tensor memory");
//   * every warp runs Alg V.2 (P:l.260-287) on TWO tiles at once (k-tiles kt, kt+1 of its stripe quadrant), their
//     steps interleaved, so a team hands the tensor core two K slices per unit step; the operand columns are double
//     buffered, so a decoder warp never waits for the tensor core in steady state;
//     (template parameter J = 1: ONE tile per warp and work item, for launches with at most one tile per team);
//   * a unit's tcgen05.st are published (wait::st, fence, mbarrier arrive) from the middle of the NEXT unit, and the unit loop
//     is unrolled by two, so that operand half, raw buffer and barrier addresses are immediates;
//   * staged lane-stream segments arrive by one cp.async.bulk per record on a per-warp mbarrier;
//   * one ISSUER warp per team (the paper's consumer warps, P:l.226-247): it sleeps on the team's "operand stored"
//     mbarrier, issues the two tcgen05.mma of the unit step (A from TMEM, X slice from shared memory, accumulator in
//     TMEM), commits them to the barrier that frees the operand columns ("ready[2]" flags of P:l.210 -> mbarriers), and
//     requests the X slices (pad16(m) rows x 32 bytes, SWIZZLE_32B) of the unit step two ahead by TMA into a 3-deep ring
//     (2-deep, one step ahead, where shared memory is short);
//   * nothing in the decode loop waits for HBM: the bf16 sign/mantissa bytes of the NEXT unit travel by cp.async into a
//     shared-memory double buffer (a register-destination global load shares scoreboards with the loop's LDS and
//     stalled every unit for an HBM round trip);
//   * the team reads its own accumulator back (tcgen05.ld: warp q -> lanes 32q..) at the end of a stripe segment;
//   * split-K: a team is a "virtual CTA" of a two-level stream-K split (pairs evenly over the CTAs, then over a CTA's
//     teams).  Every contributor of a stripe stores its partial, raises one flag per reader, waits for the flags addressed
//     to it and then reduces ITS OWN slice of the stripe's outputs, summing the contributors in team order (bit-reproducible;
//     the reduction is spread over all contributors instead of falling on one of them).
// TMEM budget: T teams x (pad16(m) accumulator columns + 32 operand columns) <= 512  ->  T = 4 up to m = 96.
#pragma once

constexpr int kTeamWarps = 4;
constexpr int kMaxTeams = 4;
constexpr int kTmemThreads = 32 * (kTeamWarps + 1) * kMaxTeams;   // 16 decoder warps + one issuer warp per team = 640: up to 96 registers
constexpr uint32_t kACols = 8;                               // TMEM columns of one operand unit (32 bytes per row)
constexpr uint32_t kASlotCols = 4 * kACols;                  // per team: two operand units (one per chain), double buffered
constexpr uint32_t kXDepth = 3;                              // X ring slots per team (each: the two slices of one unit step); 2 where shared memory is short
constexpr uint32_t kNT = 32 * kTeamWarps;                    // threads of a team

// shared-memory carve-up, from the 1024-byte aligned base: slot table | prefix scratch | barriers | X rings | raw | staging
constexpr uint32_t kTmBarOff = 16384 + 1088;                 // 64 bytes of mbarriers per team
constexpr uint32_t kTmPtrOff = kTmBarOff + 64 * kMaxTeams;
constexpr uint32_t kTmWarpBarOff = kTmPtrOff + 16;             // one mbarrier per decoder warp: its staged segments have landed
constexpr uint32_t kTmXOff = 18432;
constexpr uint32_t kRawBufBytes = 1024;                      // bf16: two 512-byte raw vectors per chain
__host__ __device__ constexpr bool tmem_has_raw(uint32_t fmt) { return fmt == ANSLIN_FMT_BF16; }
// xslices: X slices per ring slot = k-tiles per work item (2, or 1 for the kernel's J = 1)
__host__ __device__ constexpr size_t tmem_smem_bytes(uint32_t T, uint32_t mpad_max, uint32_t stream_bytes, uint32_t fmt, uint32_t xdepth = kXDepth,
                                                     uint32_t xslices = 2) {
  return 1024 /*align slack*/ + kTmXOff + size_t(T) * xdepth * xslices * mpad_max * 32 + (tmem_has_raw(fmt) ? size_t(T) * kTeamWarps * 2 * kRawBufBytes : 0) +
         size_t(T) * kTeamWarps * 2 * stream_bytes + 16;
}
// split-K control words of a problem (its flag area): u32 flag[2 * teams][PK], one word per (partial slot, reader)
constexpr size_t kTmFlagSlots = 2 * 160 * kMaxTeams;

struct TmemParams {
  Problem prob[kMaxProblems];
  uint32_t nprob;
  uint32_t T;              // teams per CTA
  uint32_t epoch;          // launch id for the split-K flags
  uint32_t stream_bytes;   // shared memory per staged lane-stream segment
  uint32_t xslice_bytes;   // max mpad * 32
  uint32_t tmem_stride;    // TMEM columns per team: max mpad + kASlotCols
  uint32_t afmt, bfmt;
  uint32_t xdepth;         // X ring slots per team: 3, or 2
};

__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]),
               "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
               : "memory");
}
__device__ __forceinline__ bool elect_one_sync() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
// Wait of a warp that has time to spare (the issuer warps): probe, then sleep.  mbarrier.try_wait's own suspension is woken
// by every barrier event of the CTA (one per ~75 clk here), and the re-probing took a sixth of the SM's issue slots.
__device__ __forceinline__ void mbar_wait_relaxed(uint32_t bar, uint32_t parity, uint32_t ns) {
  uint32_t tries = 0;
  while (!mbar_test(bar, parity)) {
    __nanosleep(ns);
    if (++tries > (1u << 24)) __trap();
  }
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
template <int KIND>  // A operand in tensor memory
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  if constexpr (KIND == 0)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
                 "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate)
                 : "memory");
  else if constexpr (KIND == 1)
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
                 "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate)
                 : "memory");
  else
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
                 "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate)
                 : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t lds16(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}

__device__ __forceinline__ void bulk_copy_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
// lane_open_segments (decode_core.cuh) for two records whose staging buffers are small enough to be copied whole without
// waiting for the segment table (bufbytes <= kTailBytes): ONE bulk copy per record, issued by lane 0 and completed on the
// warp's mbarrier `bar` (phase `parity`), instead of six 16-byte cp.async per lane and record.
// extra(): cp.async copies of the caller (first raw vectors), waited for here too.
template <class Extra, int J>
__device__ __forceinline__ void lane_open_segments_bulk(LaneStream (&s)[J], uint32_t buf0, uint32_t bufbytes, int seg, int lane, uint32_t bar,
                                                        uint32_t parity, const Extra &extra) {
  __syncwarp();   // every lane is done with the words of the previous segments
  uint32_t hdr[J], delta[J];
#pragma unroll
  for (int j = 0; j < J; ++j) {
    const uint8_t *te = s[j].rec + 4 * kLanes + kSegTableBytes * seg;
    hdr[j] = *reinterpret_cast<const uint32_t *>(te);   // u16 base | u16 total words
    delta[j] = lane < kLanes / 2 ? uint32_t(te[4 + lane]) : 0u;
  }
  if (lane == 0) {
    mbar_arrive_expect_tx(bar, uint32_t(J) * bufbytes);
#pragma unroll
    for (int j = 0; j < J; ++j) bulk_copy_g2s(buf0 + uint32_t(j) * bufbytes, s[j].rec + (s[j].goff & ~15u), bufbytes, bar);
  }
  extra();
  cp_async_commit();
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
    // the cursor is clamped into the staged buffer (see lane_open_segments)
    s[j].ptr = buf + skew + 2u * min((lane & 1) ? end_p - 1u : start_p, (bufbytes - skew) / 2u - 1u);
    s[j].goff += 2u * total;
  }
  cp_async_wait_all();
  mbar_wait(bar, parity);
#pragma unroll
  for (int j = 0; j < J; ++j) asm volatile("ld.shared.u16 %0, [%1];" : "=r"(s[j].w) : "r"(s[j].ptr) : "memory");
}

// Half H (0 / 1) of one operand unit (32 operand bytes per row = 8 registers) of the warp's two tiles: registers
// r[j][4H .. 4H+3].  rv[j]: bf16: the unit's 16 raw (sign | mantissa) bytes of this lane.  sz[j]: int4: this lane's (scale, zero)
// pair of the unit's quantisation group.  The unit is cut in two so that its housekeeping (hand-over of the previous unit,
// the next unit's raw bytes, the operand-free probe) sits between the halves, where its latencies overlap decode steps.
template <uint32_t FMT, bool PAYLOAD, int H, int J>
__device__ __forceinline__ void decode_half_regs(LaneStream (&s)[J], uint32_t tab_s, uint32_t dir, bool last_unit, const uint4 (&rv)[J],
                                                 const uint32_t (&sz)[J], uint32_t (&r)[J][8]) {
  static_assert(FMT != ANSLIN_FMT_BF16_PAIR4, "the pair variant runs on the shared-memory operand path");
  if constexpr (FMT == ANSLIN_FMT_BF16) {
    uint32_t R0[J], R1[J];
    #pragma unroll
    for (int j = 0; j < J; ++j) { R0[j] = H == 0 ? rv[j].x : rv[j].z; R1[j] = H == 0 ? rv[j].y : rv[j].w; }
    uint4 o[J];
    decode8_bf16<LaneWords, J>(s, tab_s, dir, R0, R1, o);
    if (H == 1 && PAYLOAD && last_unit) {
      // raw bytes 14, 15 of the tile's last vector ride in the END state (A4): merge them in now
#pragma unroll
      for (int j = 0; j < J; ++j) {
        const uint32_t pl = s[j].x - kL;   // byte 14 | byte 15 << 8, each = mantissa << 1 | sign
        o[j].w |= ((pl >> 1) & 0x7Fu) | ((pl & 1u) << 15) | (((pl >> 9) & 0x7Fu) << 16) | (((pl >> 8) & 1u) << 31);
      }
    }
#pragma unroll
    for (int j = 0; j < J; ++j) { r[j][4 * H] = o[j].x; r[j][4 * H + 1] = o[j].y; r[j][4 * H + 2] = o[j].z; r[j][4 * H + 3] = o[j].w; }
  } else if constexpr (FMT == ANSLIN_FMT_INT4_AWQ) {
    uint32_t Bq[J];
    decode4<LaneWords, J>(s, Bq, tab_s, dir);
#pragma unroll
    for (int j = 0; j < J; ++j) {
      const __half2 szh = *reinterpret_cast<const __half2 *>(&sz[j]);
      const __half2 sc = __half2half2(__low2half(szh));
      const __half2 zoff = __hadd2(__half2half2(__high2half(szh)), __float2half2_rn(1024.f));
      awq_dequant8(Bq[j], zoff, sc, r[j][4 * H], r[j][4 * H + 1], r[j][4 * H + 2], r[j][4 * H + 3]);
    }
  } else if constexpr (FMT == ANSLIN_FMT_FP4_E2M1) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      uint32_t Bq[J];
      decode4<LaneWords, J>(s, Bq, tab_s, dir);
#pragma unroll
      for (int j = 0; j < J; ++j) e2m1x8_to_e4m3(Bq[j], r[j][4 * H + 2 * h], r[j][4 * H + 2 * h + 1]);
    }
  } else {   // fp8 / int8: the symbol byte is the operand byte
#pragma unroll
    for (int h = 0; h < 4; ++h) {
      uint32_t q[J];
      decode4<LaneWords, J>(s, q, tab_s, dir);
#pragma unroll
      for (int j = 0; j < J; ++j) r[j][4 * H + h] = q[j];
    }
  }
}


#ifdef ANSLIN_TRACE
__device__ unsigned long long g_trace[160 * kMaxTeams * 8];
__device__ __forceinline__ unsigned long long gtimer() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define TRACE(slot) do { if (q == 0 && lane == 0) g_trace[(blockIdx.x * kMaxTeams + team) * 8 + (slot)] = gtimer(); } while (0)
__device__ unsigned long long g_prof[160 * kMaxTeams * 4 * 8];
#define PROF_DECL long long pf_t = clock64(), pf_acc[6] = {0, 0, 0, 0, 0, 0};
#define PROF(i) do { const long long pf_n = clock64(); pf_acc[i] += pf_n - pf_t; pf_t = pf_n; } while (0)
#define PROF_DUMP do { if (lane == 0) for (int pf_i = 0; pf_i < 6; ++pf_i) g_prof[((blockIdx.x * kMaxTeams + team) * 4 + q) * 8 + pf_i] = (unsigned long long)pf_acc[pf_i]; } while (0)
#define RTRACE(slot) do { if (tid == 0) g_trace[(blockIdx.x * kMaxTeams + (bar - 1)) * 8 + (slot)] = gtimer(); } while (0)
#else
#define TRACE(slot) do {} while (0)
#define RTRACE(slot) do {} while (0)
#define PROF_DECL
#define PROF(i) do {} while (0)
#define PROF_DUMP do {} while (0)
#endif

// Two-level stream-K split of the stripe-major sequence of Ptot (stripe, k-tile pair) items: first evenly over the G CTAs of
// the problem (so that every SM gets the same amount of work), then evenly over the T teams of a CTA.  Team v = c * T + t.
struct TeamMap {
  uint32_t G, T, Ptot;   // the launcher guarantees (Ptot + 1) * (G + 1) < 2^32: 32-bit arithmetic throughout
  static __device__ __forceinline__ uint32_t first_of(uint32_t c, uint32_t G, uint32_t n) { return c * n / G; }
  static __device__ __forceinline__ uint32_t owner_of(uint32_t t, uint32_t G, uint32_t n) { return ((t + 1) * G + n - 1) / n - 1; }   // largest c with first_of(c) <= t
  __device__ __forceinline__ uint32_t first(uint32_t v) const {   // first pair of team v (v = G * T: Ptot)
    const uint32_t c = v / T, t = v - c * T;
    const uint32_t a = first_of(c, G, Ptot), nc = first_of(c + 1, G, Ptot) - a;
    return a + first_of(t, T, nc);
  }
  __device__ __forceinline__ uint32_t owner(uint32_t p) const {   // the team that owns pair p
    const uint32_t c = owner_of(p, G, Ptot);
    const uint32_t a = first_of(c, G, Ptot), nc = first_of(c + 1, G, Ptot) - a;
    return c * T + owner_of(p - a, T, nc);
  }
};

// Distributed deterministic split-K reduction by one contributor team (all 128 threads) of the ns <= 2 stripes it holds a
// partial of.  The contributors of a stripe are the distinct owners of its PK pairs, in pair order; contributor vv's partial
// slot is its first segment (slot 0) unless the stripe is its second one, which can only be the case for the stripe's first
// contributor.  Every contributor sums ITS slice of the stripe's outputs over all contributors, in that order.
// Flags: a partial slot has one flag word PER READER (flags[slot * PK + reader's index among the contributors]); its writer
// sets them all to the launch epoch, every reader clears its own as soon as it has seen it, so that a replay of this very
// launch (CUDA graph: same epoch) starts from "nothing stored" without any reader counting or atomics.
// scratch: team-private shared memory, 4 * PK words.
template <uint32_t FMT, bool YB>
__device__ __forceinline__ void team_reduce(const EpiParams &p, const TeamMap &tm, uint32_t PK, int ns, const uint32_t (&stripes)[2], uint32_t v,
                                            uint32_t tid, int bar, uint32_t *scratch) {
  constexpr bool kScaled = FMT == ANSLIN_FMT_INT8 || is_fp8_path(FMT);
  uint32_t *flags = reinterpret_cast<uint32_t *>(p.counters);
  // 1. the partial slot of every pair's owner (one pair per thread)
  for (int sg = 0; sg < ns; ++sg) {
    uint32_t *list = scratch + sg * PK;
    const uint32_t p0 = stripes[sg] * PK;
    for (uint32_t k = tid; k < PK; k += kNT) {
      const uint32_t vv = tm.owner(p0 + k), v_first = tm.owner(p0);
      list[k] = vv * 2u + ((vv == v_first && tm.first(v_first) < p0) ? 1u : 0u);
    }
  }
  named_bar_sync(bar, kNT);
  // 2. how many contributors, and which one am I (consecutive pairs of one owner share a slot); thread 0 leaves the
  //    list without the repeats behind it
  uint32_t counts[2] = {1, 1}, mine[2] = {0, 0};
  for (int sg = 0; sg < ns; ++sg) {
    const uint32_t *list = scratch + sg * PK;
    uint32_t *ulist = scratch + (2 + sg) * PK;
    uint32_t count = 0, my_index = 0;
    for (uint32_t k = 0, prev = 0xFFFFFFFFu; k < PK; ++k) {
      const uint32_t sl = list[k];
      if (sl != prev) {
        if ((sl >> 1) == v) my_index = count;
        if (tid == 0) ulist[count] = sl;
        ++count;
        prev = sl;
      }
    }
    counts[sg] = count;
    mine[sg] = my_index;
  }
  // 3. wait for every contributor's flag addressed to me, and take it down
  for (int sg = 0; sg < ns; ++sg) {
    const uint32_t *list = scratch + sg * PK;
    for (uint32_t k = tid; k < PK; k += kNT) {
      if (k > 0 && list[k] == list[k - 1]) continue;
      uint32_t *flag = flags + size_t(list[k]) * PK + mine[sg];
      uint32_t val, spins = 0;
      while (true) {
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(val) : "l"(flag) : "memory");
        if (val == p.epoch) break;
        __nanosleep(100);
        if (++spins > (1u << 24)) __trap();   // a protocol bug traps instead of hanging the GPU
      }
      *reinterpret_cast<volatile uint32_t *>(flag) = 0u;
    }
  }
  RTRACE(5);
  named_bar_sync(bar, kNT);
  const size_t slot_words = size_t(p.mpad) * kTileN;
  const uint32_t n_items = p.m * 32u;   // one item = one batch row x 4 output channels
  for (int sg = 0; sg < ns; ++sg) {
    const uint32_t *ulist = scratch + (2 + sg) * PK;
    const uint32_t count = counts[sg];
    auto emit = [&](const uint32_t (&acc)[4], uint32_t it) {
      const uint32_t mm = it >> 5, n4 = stripes[sg] * kTileN + (it & 31u) * 4u;
      const float xs = kScaled ? p.x_scale[mm] : 1.0f;
      float o[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        float ws = 1.0f;
        if (FMT == ANSLIN_FMT_INT8) ws = __half2float(p.w_scale_h[n4 + j]);
        if (is_fp8_path(FMT)) ws = p.w_scale;
        o[j] = finalize<FMT>(acc[j], xs, ws);
      }
      if constexpr (YB) {
        __nv_bfloat16 *yb = reinterpret_cast<__nv_bfloat16 *>(p.y) + size_t(mm) * p.ldy + n4;
        const __nv_bfloat162 lo = __floats2bfloat162_rn(o[0], o[1]), hi = __floats2bfloat162_rn(o[2], o[3]);
        if ((reinterpret_cast<uintptr_t>(yb) & 7) == 0)
          *reinterpret_cast<uint2 *>(yb) = make_uint2(*reinterpret_cast<const uint32_t *>(&lo), *reinterpret_cast<const uint32_t *>(&hi));
        else { yb[0] = lo.x; yb[1] = lo.y; yb[2] = hi.x; yb[3] = hi.y; }
      } else {
        float *yo = p.y + size_t(mm) * p.ldy + n4;
        if ((reinterpret_cast<uintptr_t>(yo) & 15) == 0) *reinterpret_cast<float4 *>(yo) = make_float4(o[0], o[1], o[2], o[3]);
        else { yo[0] = o[0]; yo[1] = o[1]; yo[2] = o[2]; yo[3] = o[3]; }
      }
    };
    // 4. my slice of the stripe's items, two items at a time and four contributors at a time: up to eight 16-byte loads in
    //    flight per thread (the loop is bound by L2 round trips, ~1.5 us each under the launch's tail)
    const uint32_t it_begin = mine[sg] * n_items / count, it_end = (mine[sg] + 1) * n_items / count;
    for (uint32_t it = it_begin + tid; it < it_end; it += 2 * kNT) {
      const bool two = it + kNT < it_end;
      const uint32_t it1 = two ? it + kNT : it;
      const uint32_t *src0 = p.partials + size_t(it >> 5) * kTileN + (it & 31u) * 4u;
      const uint32_t *src1 = p.partials + size_t(it1 >> 5) * kTileN + (it1 & 31u) * 4u;
      uint32_t acc0[4], acc1[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) acc0[j] = acc1[j] = FMT == ANSLIN_FMT_INT8 ? 0u : __float_as_uint(0.0f);
      for (uint32_t kb = 0; kb < count; kb += 4) {
        uint4 v0[4], v1[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (kb + j < count) {
            const size_t so = size_t(ulist[kb + j]) * slot_words;
            v0[j] = ldcg128(src0 + so);
            v1[j] = ldcg128(src1 + so);
          }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {   // fixed team order -> bit-reproducible sums
          if (kb + j < count) {
            acc0[0] = acc_add<FMT>(acc0[0], v0[j].x); acc0[1] = acc_add<FMT>(acc0[1], v0[j].y);
            acc0[2] = acc_add<FMT>(acc0[2], v0[j].z); acc0[3] = acc_add<FMT>(acc0[3], v0[j].w);
            acc1[0] = acc_add<FMT>(acc1[0], v1[j].x); acc1[1] = acc_add<FMT>(acc1[1], v1[j].y);
            acc1[2] = acc_add<FMT>(acc1[2], v1[j].z); acc1[3] = acc_add<FMT>(acc1[3], v1[j].w);
          }
        }
      }
      emit(acc0, it);
      if (two) emit(acc1, it1);
    }
  }
  RTRACE(6);
}

// J = 2: a work item is a PAIR of k-tiles of one stripe, a warp interleaves the two (throughput: the default).  J = 1: a work item
// is ONE k-tile and a warp runs one chain at its latency: for launches with at most one tile per team, whose duration is the
// sequential length of an item (32 x 1024 int8 tiles of a 13824 x 5120 matrix; a 1024 x 5120 projection on its own).
template <uint32_t FMT, bool PAYLOAD, bool YB, int J = 2>
__global__ void __launch_bounds__(kTmemThreads, 1) fused_tmem_kernel(const __grid_constant__ TensorMaps tms,
                                                                      const __grid_constant__ TmemParams P) {
  using TR = FmtTraits<FMT>;
  constexpr bool kScaled = FMT == ANSLIN_FMT_INT8 || is_fp8_path(FMT);
  constexpr bool kRaw = tmem_has_raw(FMT);
  constexpr uint32_t kUnitsPerSeg = seg_steps_of(FMT) / unit_steps32(FMT);
  constexpr uint32_t kUnitK = unit_k_of(FMT);
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *smem = smem_raw + (smem0 - smem_u32(smem_raw));
  grid_dep_launch_dependents();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t T = P.T, team = uint32_t(warp) / kTeamWarps, q = uint32_t(warp) % kTeamWarps;
#ifdef ANSLIN_TRACE
  if ((threadIdx.x & 127) == 0) g_trace[(blockIdx.x * kMaxTeams + team) * 8 + 0] = gtimer();
#endif
  uint32_t pi = 0;
  while (pi + 1 < P.nprob && blockIdx.x >= P.prob[pi + 1].cta0) ++pi;
  const Problem &pr = P.prob[pi];
  // the problem's geometry, copied out of the parameter block once
  const uint8_t *const cbase = pr.cv.base;
  const uint32_t c = blockIdx.x - pr.cta0, G = pr.ncta, KT = pr.cv.KT, units = pr.cv.units, mpad = pr.mpad, tile_k = pr.cv.tile_k;
  const uint64_t off_records = pr.cv.off_records, off_raw = pr.cv.off_raw, off_scales = pr.cv.off_scales;
  const uint32_t n_out = pr.cv.n_out, qgroup = pr.cv.group;
  const CUtensorMap *const xmap = &tms.m[pi];
  uint32_t *tab = reinterpret_cast<uint32_t *>(smem);
  uint32_t *cum = reinterpret_cast<uint32_t *>(smem + 16384);
  const uint32_t bars_s = smem0 + kTmBarOff;   // per team: done[2] +0, xfull[3] +16, accfull +40, full[2] +48
  volatile uint32_t *tmemptr = reinterpret_cast<volatile uint32_t *>(smem + kTmPtrOff);
  const uint32_t XD = P.xdepth;
  const uint32_t raw_off = kTmXOff + T * XD * uint32_t(J) * P.xslice_bytes;
  const uint32_t stage_off = raw_off + (kRaw ? T * kTeamWarps * 2u * kRawBufBytes : 0u);

  // stream-K split over TEAMS (TeamMap): team v owns pairs [first(v), first(v+1)) of the stripe-major sequence of
  // (stripe, k-tile pair) items
  const uint32_t PK = (KT + J - 1) / J, stripes = n_out / kTileN, Ptot = stripes * PK;   // items per stripe
  const TeamMap tm{G, T, Ptot};
  const bool decoder = uint32_t(warp) < kTeamWarps * T;
  const uint32_t v = c * T + (decoder ? team : 0u);
  const uint32_t p_begin = tm.first(v), p_end = decoder ? tm.first(v + 1) : p_begin;
  const uint32_t *offs = reinterpret_cast<const uint32_t *>(cbase + pr.cv.off_offsets);
  // the frequency table and the record offsets of this warp's first pair of tiles: one HBM round trip for both
  const uint4 freq_regs = slot_table_load(reinterpret_cast<const uint16_t *>(cbase + pr.cv.off_freq));
  uint32_t cur_off[J] = {};
  if (p_begin < p_end) {
    const uint32_t s0 = p_begin / PK, k0 = uint32_t(J) * (p_begin % PK), t0 = (s0 * KT + k0) * 4u + q;
    cur_off[0] = offs[t0];
    if constexpr (J == 2) cur_off[1] = offs[t0 + (k0 + 1 < KT ? 4u : 0u)];
#pragma unroll
    for (int j = 0; j < J; ++j) {   // ... and the records themselves (and their raw bytes) on their way into L2
      if (lane < 24) prefetch_l2(cbase + off_records + size_t(cur_off[j]) * 16 + lane * 128);
      else if (tmem_has_raw(FMT))
        prefetch_l2(cbase + off_raw + size_t(t0 + (j && k0 + 1 < KT ? 4u : 0u)) * raw_tile_bytes(32, tile_k, PAYLOAD ? ANSLIN_FLAG_STATE_PAYLOAD : 0) + (lane - 24) * 128);
    }
  }
  if (threadIdx.x == 0) {
    for (uint32_t i = 0; i < T; ++i)
      for (uint32_t b = 0; b < 8; ++b) mbar_init(bars_s + 64 * i + 8 * b, b >= 6 ? kTeamWarps : 1);
    for (uint32_t i = 0; i < kTeamWarps * T; ++i) mbar_init(smem0 + kTmWarpBarOff + 8 * i, 1);
    fence_mbar_init();
  }
  if (warp == 0) tmem_alloc(smem0 + kTmPtrOff, 512);
  tc_fence_before();
  build_slot_table(tab, cum, freq_regs);   // ends with __syncthreads()
  tc_fence_after();
  const uint32_t tmem_base = *tmemptr;

  const uint32_t done_s = bars_s + 64 * team, accfull_s = done_s + 40, full_s = done_s + 48;
  const uint32_t acc_t = tmem_base + team * P.tmem_stride, a_t = acc_t + mpad;   // accumulator, then two operand units
  const uint32_t lane_t = (q * 32u) << 16;
  const uint32_t rawbuf_s = smem0 + raw_off + uint32_t(warp) * 2u * kRawBufBytes;  // chain j, vector parity b at j * 1024 + b * 512
  const uint32_t rawlane_s = rawbuf_s + 16u * uint32_t(lane);                        // ... this lane's 16 bytes of it
  const uint32_t stage_s = smem0 + stage_off + uint32_t(warp) * 2u * P.stream_bytes, tab_s = smem0;
  const uint32_t dir = (lane & 1) ? uint32_t(-2) : 2u;
  const int bar_id = 1 + int(team);


  const EpiParams ep{pr.x_scale, reinterpret_cast<const __half *>(cbase + off_scales), pr.cv.w_scale, pr.y, pr.ldy,
                     pr.partials, pr.counters, P.epoch, pr.m, mpad};
  const uint32_t idesc = make_idesc(TR::c, P.afmt, P.bfmt, 128, mpad);
  const uint32_t xbytes = mpad * 32u;
  const size_t rtb = raw_tile_bytes(32, tile_k, PAYLOAD ? ANSLIN_FLAG_STATE_PAYLOAD : 0);
  uint32_t fin_stripe[2] = {0, 0};
  bool fin_valid[2] = {false, false};

  if (uint32_t(warp) >= kTeamWarps * T) {
    // ===================== issuer warp of team `it`: drives the tensor core and the team's X ring =====================
    // Every wait is a hardware-suspended mbarrier wait, so this warp costs the decoders next to nothing, and the MMAs and
    // TMA requests of a unit step cost the decoder warps nothing at all.
    const uint32_t it = uint32_t(warp) - kTeamWarps * T, vt = c * T + it;
    const uint32_t pb = tm.first(vt), pe = tm.first(vt + 1), Nt = (pe - pb) * units;
    const uint32_t bt = bars_s + 64 * it, acc = tmem_base + it * P.tmem_stride, at = acc + mpad;
    const uint32_t xr = smem0 + kTmXOff + it * XD * uint32_t(J) * P.xslice_bytes;   // ring slot sx, slice j at (sx * J + j) * xslice_bytes
    const uint64_t bdesc0 = make_smem_desc(xr, 16, 256, kLayoutSW32);
    const uint32_t bdesc_step = P.xslice_bytes >> 4;
    const bool leader = elect_one_sync();
    uint32_t kpx = pb % PK, ux = 0, sxx = 0, nx = 0;   // X request cursor: pair in stripe, unit, ring slot, unit step
    auto request_x = [&]() {   // the two X slices of unit step nx
      if (leader) {
        const uint32_t ktA = uint32_t(J) * kpx, bar = bt + 16 + 8 * sxx;
        const bool hasB = J == 2 && ktA + 1 < KT;
        const int kA = int(ktA * tile_k + ux * kUnitK);
        mbar_arrive_expect_tx(bar, hasB ? 2 * xbytes : xbytes);
        tma_load_2d(xr + (sxx * uint32_t(J)) * P.xslice_bytes, xmap, kA, 0, bar);
        if (hasB) tma_load_2d(xr + (sxx * uint32_t(J) + 1u) * P.xslice_bytes, xmap, kA + int(tile_k), 0, bar);
      }
      ++nx;
      if (++sxx == XD) sxx = 0;
      if (++ux == units) { ux = 0; if (++kpx == PK) kpx = 0; }
    };
    grid_dep_wait();   // X belongs to the stream's earlier kernels until they are done
    for (uint32_t i = 0; i + 1 < XD && i < Nt; ++i) request_x();   // XD - 1 unit steps ahead
    uint32_t pp = pb, kp = pb % PK, u = 0, sx = 0, xpar = 0;
#pragma unroll 1
    for (uint32_t n = 0; n < Nt; ++n) {
      const uint32_t sa = n & 1u;
      mbar_wait_relaxed(bt + 48 + 8 * sa, (n >> 1) & 1u, 250);   // all four decoder warps have stored this step's operand columns
      mbar_wait_relaxed(bt + 16 + 8 * sx, xpar, 100);            // its X slices have landed
      tc_fence_after();
      const bool hasB = J == 2 && 2u * kp + 1 < KT, last_unit = u + 1 == units;
      const bool seg_first = u == 0 && (pp == pb || kp == 0), seg_last = last_unit && (pp + 1 == pe || kp + 1 == PK);
      if (leader) {
        const uint64_t bdA = bdesc0 + uint64_t(sx * uint32_t(J) * bdesc_step);
        umma_ts<TR::kind>(acc, at + sa * 2u * kACols, bdA, idesc, seg_first ? 0u : 1u);
        if (hasB) umma_ts<TR::kind>(acc, at + sa * 2u * kACols + kACols, bdA + bdesc_step, idesc, 1u);
        umma_commit(bt + 8 * sa);
        if (seg_last) umma_commit(bt + 40);
      }
      __syncwarp();
      if (++sx == XD) { sx = 0; xpar ^= 1u; }
      if (last_unit) { u = 0; ++pp; if (++kp == PK) kp = 0; } else ++u;
      // the X slices of step n + XD - 1 go to the ring slot last read by the MMAs of step n - 1 (issued one step ago)
      if (nx < Nt) {
        if (n >= 1) mbar_wait_relaxed(bt + 8 * ((n - 1) & 1u), ((n - 1) >> 1) & 1u, 100);
        request_x();
      }
    }
  } else {
  uint32_t seg_i = 0;
#ifdef ANSLIN_TRACE
  uint32_t n = 0;
#endif
  bool dep_waited = false;
#ifdef ANSLIN_SKEL_NO_RAW   // timing experiment only (wrong results): how much does the raw-byte path cost
  constexpr bool kRawOn = false;
#else
  constexpr bool kRawOn = kRaw;
#endif
  // hand-over of a unit step, second part: wait for the warp's tensor-memory stores, then the arrival that (as the fourth of
  // the team) lets the issuer warp multiply the step.  Deferred to the middle of the next unit so that the store latency
  // overlaps decode steps; completed before anything waits for the step's MMAs (the segment's epilogue).
  bool pending = false;       // a unit's stores are not yet published
  uint32_t open_par = 0;      // phase of the warp's staging barrier
  const uint32_t warpbar_s = smem0 + kTmWarpBarOff + 8u * uint32_t(warp);
  uint32_t kpar = 0;          // parity of (unit step / 2): the phase of the operand-free barriers
  auto finish_handover = [&](uint32_t full_bar) {
    if (pending) {
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(full_bar);
      pending = false;
    }
  };
  // Teams start half a microsecond apart: the sixteen decoder warps of an SM otherwise run in lock step, and every tile opening
  // and hand-over of one team then coincides with the others'.  The offset persists for the launch and pays for itself
  // (0.2800 against 0.2820 ms per step; 1 us apart the same, 1.5 us apart 0.2843: profiles/r2_skeleton_experiments.md).
#ifndef ANSLIN_STAGGER_NS
#define ANSLIN_STAGGER_NS 500
#endif
  __nanosleep(team * ANSLIN_STAGGER_NS);
  TRACE(1);
  PROF_DECL
#pragma unroll 1
  for (uint32_t p = p_begin; p < p_end; ++seg_i) {
    const uint32_t stripe = p / PK, kp0 = p % PK, np = min(PK - kp0, p_end - p);
    const bool whole = kp0 == 0 && np == PK;
#pragma unroll 1
    for (uint32_t i = 0; i < np; ++i) {
      const uint32_t ktA = uint32_t(J) * (kp0 + i);
      const bool hasB = J == 2 && ktA + 1 < KT;
      LaneStream s[J];
      uint32_t tile[J];
      tile[0] = (stripe * KT + ktA) * 4u + q;
      if constexpr (J == 2) tile[1] = hasB ? tile[0] + 4u : tile[0];   // odd KT: the second chain re-decodes the first tile; its output is never multiplied
      const uint8_t *rawp[J] = {};   // this lane's 16 bytes of the NEXT raw vector to fetch
#pragma unroll
      for (int j = 0; j < J; ++j) {
        const uint8_t *rec = cbase + off_records + size_t(cur_off[j]) * 16;
        lane_open(s[j], rec, int(units / kUnitsPerSeg), lane);
        if (kRaw) rawp[j] = cbase + off_raw + size_t(tile[j]) * rtb + 16 * lane;
      }
      // the records of this warp's next pair: pulled into L2 during the first unit
      const bool has_next = p + i + 1 < p_end;
      uint32_t next_tile = 0, next_off[J] = {};
      if (has_next) {
        const uint32_t pn = p + i + 1, sn = pn / PK, kn = uint32_t(J) * (pn % PK);
        next_tile = (sn * KT + kn) * 4u + q;
        next_off[0] = offs[next_tile];
        if constexpr (J == 2) next_off[1] = offs[next_tile + (kn + 1 < KT ? 4u : 0u)];
      }
      uint32_t sz_cur[J] = {}, sz_left = 0;   // int4: the current (scale, zero) pairs and the units they still hold for
      // One unit of both tiles.  A tile has an even number of units (tmem_eligible), so the parity PAR of a unit step — which
      // half of the operand columns, which raw buffer, which barriers — is a compile-time constant of each copy of the body.
      auto unit_body = [&](auto par_c, const uint32_t u) {
        constexpr uint32_t PAR = decltype(par_c)::value;
        if constexpr (PAR == 1) {
          if (u == 1 && has_next) {
#pragma unroll
            for (int j = 0; j < J; ++j) {
              if (lane < 24) prefetch_l2(cbase + off_records + size_t(next_off[j]) * 16 + lane * 128);
              else if (kRaw) prefetch_l2(cbase + off_raw + size_t(next_tile + 4u * uint32_t(j)) * rtb + (lane - 24) * 128);
              cur_off[j] = next_off[j];   // the next pair opens without another look at the offset table
            }
          }
        } else {
          if (u == 0) PROF(6);
          if (u % kUnitsPerSeg == 0) {
            // stage the segment (drains cp.async first and last); at the tile's start its first raw vector rides in the same group
            auto first_raw = [&]() {
              if (kRawOn && u == 0) {
#pragma unroll
                for (int j = 0; j < J; ++j) { cp_async16(rawlane_s + uint32_t(j) * kRawBufBytes, rawp[j]); rawp[j] += 512; }
              }
            };
            if (P.stream_bytes <= uint32_t(kTailBytes)) {
              lane_open_segments_bulk(s, stage_s, P.stream_bytes, int(u / kUnitsPerSeg), lane, warpbar_s, open_par, first_raw);
              open_par ^= 1u;
            } else {
              lane_open_segments<J>(s, stage_s, P.stream_bytes, int(u / kUnitsPerSeg), lane, first_raw);
            }
          }
          if (u == 0) PROF(4);
          if (!dep_waited) {   // everything before this point read the container only
            grid_dep_wait();
            dep_waited = true;
          }
        }
        const bool last_unit = PAR == 1 && u + 1 == units;
        uint4 rv[J];
        uint32_t sz[J];
#pragma unroll
        for (int j = 0; j < J; ++j) { rv[j] = make_uint4(0, 0, 0, 0); sz[j] = 0; }
        if constexpr (kRawOn) {
          // this unit's raw vector was copied during the previous unit; fetch the next one into the other buffer.
          // rawp[j]: at an even unit the next vector, at an odd unit the one before it (advanced by two vectors at a time)
          PROF(0);
          cp_async_wait_all();
          PROF(7);
          const uint32_t rb = rawlane_s + PAR * 512u;
          if (PAYLOAD && last_unit) {
            // last vector with the state-payload flag: 7 sub-rows of 32 x 2 bytes (bytes 14, 15 come from the end state)
            __syncwarp();
#pragma unroll
            for (int j = 0; j < J; ++j) {
              uint32_t h[7];
#pragma unroll
              for (int k = 0; k < 7; ++k)
                h[k] = lds16(rawbuf_s + 512u + uint32_t(j) * kRawBufBytes + uint32_t(k) * 64u + 2u * uint32_t(lane));
              rv[j] = make_uint4(h[0] | (h[1] << 16), h[2] | (h[3] << 16), h[4] | (h[5] << 16), h[6]);
            }
          } else {
#pragma unroll
            for (int j = 0; j < J; ++j) rv[j] = lds128(rb + uint32_t(j) * kRawBufBytes);
          }
          if (!last_unit) {
            const bool short_vec = PAYLOAD && PAR == 0 && u + 2 == units;   // the next vector is the payload-shortened one: 448 bytes
            if (!short_vec || lane < 28) {
#pragma unroll
              for (int j = 0; j < J; ++j) cp_async16(rawlane_s + uint32_t(j) * kRawBufBytes + (PAR ^ 1u) * 512u, rawp[j] + PAR * 512u);
            }
            cp_async_commit();
          }
          if constexpr (PAR == 1) {
#pragma unroll
            for (int j = 0; j < J; ++j) rawp[j] += 1024;
          }
        }
        if constexpr (FMT == ANSLIN_FMT_INT4_AWQ) {
          // this lane's (scale, zero) pairs: loaded again only where a tile's k range enters another quantisation group
          if (sz_left == 0) {
            sz_left = 0xFFFFFFFFu;
#pragma unroll
            for (int j = 0; j < J; ++j) {
              const uint32_t k_elem = (ktA + uint32_t(j)) * tile_k + u * kUnitK;
              sz_cur[j] = __ldg(reinterpret_cast<const uint32_t *>(cbase + off_scales) + size_t(k_elem / qgroup) * n_out + size_t(stripe) * kTileN +
                                q * 32u + uint32_t(lane));
              sz_left = min(sz_left, (qgroup - k_elem % qgroup) / kUnitK);   // units until chain j's next group (group sizes are multiples of 16)
            }
          }
          --sz_left;
#pragma unroll
          for (int j = 0; j < J; ++j) sz[j] = sz_cur[j];
        }
        // have the MMAs that read this half of the operand columns two steps ago finished?  (On fresh barriers the parity
        // of the "previous" phase passes at once.)  Asked now, needed after the unit is decoded.
        const bool slot_free = mbar_test(done_s + 8 * PAR, kpar ^ 1u);
        uint32_t r[J][8];
#ifdef ANSLIN_TRACE
        if (blockIdx.x == 7 && lane == 0 && n + PAR < 48) g_prof[160 * kMaxTeams * 4 * 8 - 4 * 4 * 48 + ((team * 4 + q) * 48 + n + PAR)] = gtimer();
#endif
        PROF(0);
#ifdef ANSLIN_SKEL_NO_DECODE   // timing experiment only (wrong results): everything but the rANS steps
#pragma unroll
        for (int k = 0; k < 8; ++k) { r[0][k] = rv[0].x + k; r[J - 1][k] = rv[J - 1].y ^ k; }
        finish_handover(full_s + 8 * (PAR ^ 1u));
#else
        decode_half_regs<FMT, PAYLOAD, 0>(s, tab_s, dir, last_unit, rv, sz, r);
        // the PREVIOUS unit's tensor-memory stores have had half a unit to land: publish them now, between the halves
        finish_handover(full_s + 8 * (PAR ^ 1u));
        decode_half_regs<FMT, PAYLOAD, 1>(s, tab_s, dir, last_unit, rv, sz, r);
#endif
        PROF(1);
        // ---- hand-over: registers -> tensor memory (-> tcgen05.mma once the stores are published) ----
        if (!slot_free) mbar_wait(done_s + 8 * PAR, kpar ^ 1u);
        PROF(2);
#ifdef ANSLIN_SKEL_NO_STTM   // timing experiment only (wrong results): how much do the tensor-memory stores cost
        if (r[0][0] == 0x12345678u && r[J - 1][7] == 0x9abcdef0u && r[0][3] == 1u && r[J - 1][2] == 7u) {
#endif
        tmem_st8(a_t + PAR * 2u * kACols + lane_t, r[0]);
        if constexpr (J == 2) tmem_st8(a_t + PAR * 2u * kACols + kACols + lane_t, r[J - 1]);
#ifdef ANSLIN_SKEL_NO_STTM
        }
#endif
        pending = true;
        PROF(3);
      };
#pragma unroll 1
      for (uint32_t u = 0; u < units; u += 2) {
        unit_body(std::integral_constant<uint32_t, 0>{}, u);
        unit_body(std::integral_constant<uint32_t, 1>{}, u + 1);
        kpar ^= 1u;
#ifdef ANSLIN_TRACE
        n += 2;
#endif
      }
#ifdef ANSLIN_BOUNDS_CHECK   // debug builds (compute-sanitizer is closed on this pool): every word cursor ended inside its staged buffer
#pragma unroll
      for (int j = 0; j < J; ++j) {
        const uint32_t lo = stage_s + uint32_t(j) * P.stream_bytes;
        if (s[j].ptr + 2u < lo || s[j].ptr > lo + P.stream_bytes) __trap();
        if (PAYLOAD && (s[j].x < kL || s[j].x >= 2u * kL)) __trap();   // the end state is L + payload
        if (!PAYLOAD && s[j].x != kL) __trap();                        // ... or exactly the encoder's start state
      }
#endif
    }
    finish_handover(full_s + 8);   // a tile ends with an odd unit
    PROF(0);
    // ---- epilogue of this stripe segment: the team reads its own accumulator ----
    TRACE(2);
    mbar_wait(accfull_s, seg_i & 1u);
    TRACE(3);
    tc_fence_after();
    {
      const uint32_t row = q * 32u + uint32_t(lane), nrow = stripe * kTileN + row;
      float ws = 1.0f;
      if (FMT == ANSLIN_FMT_INT8) ws = __half2float(ep.w_scale_h[nrow]);
      if (is_fp8_path(FMT)) ws = ep.w_scale;
      const uint32_t seg = (p == p_begin ? 0u : 1u);
      uint32_t *part = ep.partials + size_t(v * 2u + seg) * mpad * kTileN;
      for (uint32_t c0 = 0; c0 < mpad; c0 += 16) {
        uint32_t val[16];
        tmem_ld16(acc_t + lane_t + c0, val);
        if (whole) {
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            const uint32_t mm = c0 + j;
            if (mm < ep.m) {
              const float f = finalize<FMT>(val[j], kScaled ? ep.x_scale[mm] : 1.0f, ws);
              if constexpr (YB) reinterpret_cast<__nv_bfloat16 *>(ep.y)[size_t(mm) * ep.ldy + nrow] = __float2bfloat16_rn(f);
              else ep.y[size_t(mm) * ep.ldy + nrow] = f;
            }
          }
        } else {   // the partial buffer has mpad rows: no guards
#pragma unroll
          for (int j = 0; j < 16; ++j) part[size_t(c0 + j) * kTileN + row] = val[j];
        }
      }
      tc_fence_before();   // the next segment's first MMA (after the next team barrier) overwrites the accumulator
      if (!whole) {
        // the team's partial stores are ordered before the barrier; the release store of a thread that raises a flag is
        // cumulative over what the barrier made visible to it (no separate fence: st.release.gpu carries it)
        named_bar_sync(bar_id, kNT);
        {   // one flag per possible reader of this partial (team_reduce)
          uint32_t *flag = reinterpret_cast<uint32_t *>(ep.counters) + size_t(v * 2u + seg) * PK;
          for (uint32_t rdr = q * 32u + uint32_t(lane); rdr < PK; rdr += kNT)
            asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(flag + rdr), "r"(ep.epoch) : "memory");
        }
        if (seg == 0) { fin_stripe[0] = stripe; fin_valid[0] = true; }
        else { fin_stripe[1] = stripe; fin_valid[1] = true; }
      }
    }
    PROF(5);
    p += np;
  }
  PROF_DUMP;
  cp_async_wait_all();
  TRACE(4);
  // ---- split-K: reduce this team's slice of every stripe it holds a partial of ----
  if (!dep_waited) grid_dep_wait();
  const uint32_t tid = q * 32u + uint32_t(lane);
  if (fin_valid[0] || fin_valid[1]) {
    named_bar_sync(bar_id, kNT);   // the scratch below is the staging area the team's warps decoded from
    uint32_t st[2] = {fin_valid[0] ? fin_stripe[0] : fin_stripe[1], fin_stripe[1]};
    team_reduce<FMT, YB>(ep, tm, PK, (fin_valid[0] && fin_valid[1]) ? 2 : 1, st, v, tid, bar_id,
                         reinterpret_cast<uint32_t *>(smem + stage_off + size_t(team) * kTeamWarps * 2u * P.stream_bytes));
  }
  TRACE(7);
  }   // decoder warps
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem_base, 512);
}
