// Decode-only kernel for lane-stream containers with 32-row tiles (anslin_decode; the paper's unfused stage, Fig. 9 P:l.410).
// Included by kernels.cu after fused_tmem.cuh, whose decoder-side pieces it reuses (decode_half_regs, the bulk-copy segment
// opening, the cp.async raw-byte double buffer, the unit loop unrolled by two).
//   * 16 decoder warps per CTA, one CTA per SM, every warp Alg V.2 (P:l.260-287) on TWO tiles at once (tiles 2j, 2j + 1 of
//     the container: two row quadrants of one (stripe, k-tile) group);
//   * lane l is row l of its tile: the 32 bytes of row-major W it decodes per unit go from registers into a 32 x 32-byte
//     shared-memory box, and ONE elected lane hands the box to the TMA store engine (cp.async.bulk.tensor, shared -> global):
//     no per-lane global store instruction, no transposition through shared memory, nothing on the LSU pipe but two STS.128
//     per lane and unit (a lane-per-row STG.128 costs one L1 wavefront per row: 64 per unit and chain);
//   * the boxes are double buffered per chain; cp.async.bulk.wait_group.read frees a box two units later.
// Formats: bf16 (16 weights = 32 bytes per row and unit), int8 / fp8 (32 weights), and the packed 4-bit formats in their stored
// packing (fp4: 16 bytes per unit; int4: 8, two units per box row).  128-row tiles, interleaved words and the bf16 pair variant
// stay on decode_kernel.
#pragma once

constexpr int kLaneDecWarps = 16;
__host__ __device__ constexpr bool decode_lanes_format(uint32_t fmt) {
  return fmt == ANSLIN_FMT_BF16 || fmt == ANSLIN_FMT_INT8 || is_fp8(fmt) || is_packed4(fmt);
}
// bytes of row-major W a lane decodes per unit (bf16: 16 weights, int8 / fp8: 32, fp4: 32 codes = 16 bytes, int4: 16 codes = 8 bytes)
// and bytes per box row: the TMA engine wants at least 16, so an int4 box row holds two units
__host__ __device__ constexpr uint32_t decode_lanes_unit_bytes(uint32_t fmt) { return fmt == ANSLIN_FMT_INT4_AWQ ? 8u : fmt == ANSLIN_FMT_FP4_E2M1 ? 16u : 32u; }
__host__ __device__ constexpr uint32_t decode_lanes_box_row(uint32_t fmt) { return is_packed4(fmt) ? 16u : 32u; }
// shared memory from the 1024-byte aligned base: slot table 16 KiB | prefix scratch + warp barriers 2 KiB | per warp: raw 2 KiB
// (bf16 only) | four out boxes (two chains, double buffered) | two staged segments
__host__ __device__ constexpr uint32_t decode_lanes_raw_bytes(uint32_t fmt) { return fmt == ANSLIN_FMT_BF16 ? 2u * kRawBufBytes : 0u; }
__host__ __device__ constexpr uint32_t decode_lanes_box_bytes(uint32_t fmt) { return 32u * decode_lanes_box_row(fmt); }
__host__ __device__ constexpr size_t decode_lanes_smem(uint32_t fmt, uint32_t warps, uint32_t stream_bytes) {
  return 1024 + 18432 + size_t(warps) * (decode_lanes_raw_bytes(fmt) + 4 * decode_lanes_box_bytes(fmt) + 2 * size_t(stream_bytes)) + 16;
}

__device__ __forceinline__ void tma_store_2d(const CUtensorMap *map, uint32_t src, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(map), "r"(src), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }

template <uint32_t FMT, bool PAYLOAD>
__global__ void __launch_bounds__(kLaneDecWarps * 32, 1) decode_lanes_kernel(const __grid_constant__ CUtensorMap tmo, const ContainerView cv,
                                                                             const uint32_t stream_bytes) {
  constexpr bool kRaw = FMT == ANSLIN_FMT_BF16;
  constexpr uint32_t kUnitsPerSeg = seg_steps_of(FMT) / unit_steps32(FMT);
  constexpr uint32_t kUB = decode_lanes_unit_bytes(FMT);
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem0 = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t *smem = smem_raw + (smem0 - smem_u32(smem_raw));
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t W = blockDim.x >> 5, G = gridDim.x, KT = cv.KT, units = cv.units;
  const uint8_t *const cbase = cv.base;
  uint32_t *tab = reinterpret_cast<uint32_t *>(smem);
  uint32_t *cum = reinterpret_cast<uint32_t *>(smem + 16384);
  // jobs (pairs of consecutive tiles) evenly over the CTAs, then over a CTA's warps
  const uint32_t jobs = cv.n_tiles / 2;
  const uint32_t ja = uint32_t(uint64_t(blockIdx.x) * jobs / G), jn = uint32_t(uint64_t(blockIdx.x + 1) * jobs / G) - ja;
  const uint32_t j_begin = ja + uint32_t(warp) * jn / W, j_end = ja + uint32_t(warp + 1) * jn / W;
  const uint32_t *offs = reinterpret_cast<const uint32_t *>(cbase + cv.off_offsets);
  // programmatic dependent launch: this CTA may have been scheduled under the previous kernel's tail; the container (which that
  // kernel may have written: anslin_encode_device) is not touched before it is complete
  grid_dep_launch_dependents();
  grid_dep_wait();
  const uint4 freq_regs = slot_table_load(reinterpret_cast<const uint16_t *>(cbase + cv.off_freq));
  uint32_t cur_off[2] = {0, 0};
  if (j_begin < j_end) { cur_off[0] = offs[2 * j_begin]; cur_off[1] = offs[2 * j_begin + 1]; }
  const uint32_t warpbar_s = smem0 + 16384 + 1088 + 8u * uint32_t(warp);
  if (threadIdx.x == 0) {
    for (uint32_t i = 0; i < W; ++i) mbar_init(smem0 + 16384 + 1088 + 8 * i, 1);
    fence_mbar_init();
  }
  build_slot_table(tab, cum, freq_regs);   // ends with __syncthreads()

  const uint32_t tab_s = smem0, per_warp0 = smem0 + 18432;
  constexpr uint32_t kRawBytes = decode_lanes_raw_bytes(FMT), kOutBoxBytes = decode_lanes_box_bytes(FMT);
  const uint32_t rawbuf_s = per_warp0 + uint32_t(warp) * kRawBytes, rawlane_s = rawbuf_s + 16u * uint32_t(lane);
  const uint32_t out_s = per_warp0 + W * kRawBytes + uint32_t(warp) * 4u * kOutBoxBytes;   // box (chain j, parity b) at (j * 2 + b) boxes
  const uint32_t stage_s = per_warp0 + W * (kRawBytes + 4u * kOutBoxBytes) + uint32_t(warp) * 2u * stream_bytes;
  const uint32_t dir = (lane & 1) ? uint32_t(-2) : 2u;
  const size_t rtb = raw_tile_bytes(32, cv.tile_k, PAYLOAD ? ANSLIN_FLAG_STATE_PAYLOAD : 0);
  const uint32_t tile_row_bytes = uint32_t(row_bytes_of(FMT, cv.tile_k));
  // a lane's two 16-byte halves of its row go to the box in an order that keeps the stores free of bank conflicts
  const bool swap_halves = (lane >> 2) & 1;
  const uint32_t box_lane = uint32_t(lane) * 32u;
  uint32_t open_par = 0;

#pragma unroll 1
  for (uint32_t job = j_begin; job < j_end; ++job) {
    const uint32_t t0 = 2u * job, grp = t0 >> 2, q0 = t0 & 3u, stripe = grp / KT, kt = grp % KT;
    LaneStream s[2];
    const uint8_t *rawp[2] = {nullptr, nullptr};
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      lane_open(s[j], cbase + cv.off_records + size_t(cur_off[j]) * 16, int(units / kUnitsPerSeg), lane);
      if (kRaw) rawp[j] = cbase + cv.off_raw + size_t(t0 + uint32_t(j)) * rtb + 16 * lane;
    }
    const int row0 = int(stripe * kTileN + q0 * 32u), col0 = int(kt * tile_row_bytes);
    const bool has_next = job + 1 < j_end;
    uint32_t next_off[2] = {0, 0};
    if (has_next) { next_off[0] = offs[t0 + 2]; next_off[1] = offs[t0 + 3]; }
    auto unit_body = [&](auto par_c, const uint32_t u) {
      constexpr uint32_t PAR = decltype(par_c)::value;
      if constexpr (PAR == 1) {
        if (u == 1 && has_next) {   // the next job's records and raw bytes on their way into L2
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            if (lane < 24) prefetch_l2(cbase + cv.off_records + size_t(next_off[j]) * 16 + lane * 128);
            else if (kRaw) prefetch_l2(cbase + cv.off_raw + size_t(t0 + 2u + uint32_t(j)) * rtb + (lane - 24) * 128);
            cur_off[j] = next_off[j];
          }
        }
      } else {
        if (u % kUnitsPerSeg == 0) {
          auto first_raw = [&]() {
            if (kRaw && u == 0) {
#pragma unroll
              for (int j = 0; j < 2; ++j) { cp_async16(rawlane_s + uint32_t(j) * kRawBufBytes, rawp[j]); rawp[j] += 512; }
            }
          };
          if (stream_bytes <= uint32_t(kTailBytes)) {
            lane_open_segments_bulk(s, stage_s, stream_bytes, int(u / kUnitsPerSeg), lane, warpbar_s, open_par, first_raw);
            open_par ^= 1u;
          } else {
            lane_open_segments<2>(s, stage_s, stream_bytes, int(u / kUnitsPerSeg), lane, first_raw);
          }
        }
      }
      const bool last_unit = PAR == 1 && u + 1 == units;
      uint4 rv[2] = {make_uint4(0, 0, 0, 0), make_uint4(0, 0, 0, 0)};
      const uint32_t sz[2] = {0, 0};
      if constexpr (kRaw) {   // as in fused_tmem_kernel: this unit's raw vector was copied during the previous unit
        cp_async_wait_all();
        if (PAYLOAD && last_unit) {
          __syncwarp();
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            uint32_t h[7];
#pragma unroll
            for (int k = 0; k < 7; ++k) h[k] = lds16(rawbuf_s + 512u + uint32_t(j) * kRawBufBytes + uint32_t(k) * 64u + 2u * uint32_t(lane));
            rv[j] = make_uint4(h[0] | (h[1] << 16), h[2] | (h[3] << 16), h[4] | (h[5] << 16), h[6]);
          }
        } else {
#pragma unroll
          for (int j = 0; j < 2; ++j) rv[j] = lds128(rawlane_s + PAR * 512u + uint32_t(j) * kRawBufBytes);
        }
        if (!last_unit) {
          const bool short_vec = PAYLOAD && PAR == 0 && u + 2 == units;
          if (!short_vec || lane < 28) {
#pragma unroll
            for (int j = 0; j < 2; ++j) cp_async16(rawlane_s + uint32_t(j) * kRawBufBytes + (PAR ^ 1u) * 512u, rawp[j] + PAR * 512u);
          }
          cp_async_commit();
        }
        if constexpr (PAR == 1) { rawp[0] += 1024; rawp[1] += 1024; }
      }
      uint32_t r[2][8];
      if constexpr (is_packed4(FMT)) {   // the stored packing: one coded byte = two 4-bit codes
#pragma unroll
        for (int h = 0; h < int(kUB / 4); ++h) {
          uint32_t Bq[2];
          decode4<LaneWords, 2>(s, Bq, tab_s, dir);
          r[0][h] = Bq[0];
          r[1][h] = Bq[1];
        }
      } else {
        decode_half_regs<FMT, PAYLOAD, 0>(s, tab_s, dir, last_unit, rv, sz, r);
        decode_half_regs<FMT, PAYLOAD, 1>(s, tab_s, dir, last_unit, rv, sz, r);
      }
      // ---- registers -> shared-memory box -> TMA store ----
      // box parity: the unit's (one box per unit) or the unit pair's (int4: two units fill one box row)
      const uint32_t bpar = kUB == 8 ? ((u >> 1) & 1u) : PAR;
      const bool first_of_box = kUB != 8 || PAR == 0, last_of_box = kUB != 8 || PAR == 1;
      if (first_of_box) {
        if (lane == 0) bulk_wait_read<1>();   // the stores that last used this parity's boxes have read them
        __syncwarp();
      }
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const uint32_t box0 = out_s + (uint32_t(j) * 2u + bpar) * kOutBoxBytes;
        if constexpr (kUB == 32) {
          const uint32_t box = box0 + box_lane;
          const uint4 lo = make_uint4(r[j][0], r[j][1], r[j][2], r[j][3]), hi = make_uint4(r[j][4], r[j][5], r[j][6], r[j][7]);
          sts128(box + (swap_halves ? 16u : 0u), swap_halves ? hi : lo);
          sts128(box + (swap_halves ? 0u : 16u), swap_halves ? lo : hi);
        } else if constexpr (kUB == 16) {
          sts128(box0 + uint32_t(lane) * 16u, make_uint4(r[j][0], r[j][1], r[j][2], r[j][3]));
        } else {
          asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(box0 + uint32_t(lane) * 16u + PAR * 8u), "r"(r[j][0]), "r"(r[j][1]) : "memory");
        }
      }
      if (last_of_box) {
        fence_proxy_async();   // generic-proxy stores -> visible to the TMA engine's async proxy
        __syncwarp();
        if (lane == 0) {
          const int col = col0 + int((kUB == 8 ? (u & ~1u) : u) * kUB);
#pragma unroll
          for (int j = 0; j < 2; ++j) tma_store_2d(&tmo, out_s + (uint32_t(j) * 2u + bpar) * kOutBoxBytes, col, row0 + 32 * j);
          bulk_commit();
        }
      }
    };
#pragma unroll 1
    for (uint32_t u = 0; u < units; u += 2) {
      unit_body(std::integral_constant<uint32_t, 0>{}, u);
      unit_body(std::integral_constant<uint32_t, 1>{}, u + 1);
    }
#ifdef ANSLIN_BOUNDS_CHECK   // debug builds (compute-sanitizer is closed on this pool): every word cursor ended inside its staged buffer
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const uint32_t lo = stage_s + uint32_t(j) * stream_bytes;
      if (s[j].ptr + 2u < lo || s[j].ptr > lo + stream_bytes) __trap();
      if (PAYLOAD && (s[j].x < kL || s[j].x >= 2u * kL)) __trap();   // the end state is L + payload
      if (!PAYLOAD && s[j].x != kL) __trap();                        // ... or exactly the encoder's start state
    }
#endif
  }
  cp_async_wait_all();
  if (lane == 0) bulk_wait_read<0>();   // the boxes stay valid until the engine has read them
}
