// GPU-side encoder (S: §8(f) NEXT-6; P:l.486 names it as future work): compress a row-major weight tensor that is
// already resident in HBM into a lane-stream container (32-row tiles) in HBM, without a round trip of W through the host.
// Only a 4 KiB histogram and the per-tile record sizes visit the host (table normalisation and the offset prefix sum).
//
//   1. anslin_histogram            256-bin counts of the coded symbols             (device, one pass over W)
//   2. normalise_freqs             12-bit frequency table, A10            (host, 256 entries)
//   3. enc_count_kernel            every lane runs its rANS encoder in reverse and counts the 16-bit words it would emit per
//                                  256-step segment -> record sizes, segment tables (device)
//   4. exclusive sum of sizes      record offsets                                    (host, 4 bytes per tile)
//   5. enc_write_kernel            the same encoder pass again, now storing every word at its final address: lane 2p's
//                                  words ascending from its region start, lane 2p+1's descending from the region end
//                                  (the encoder emits in reverse read order); states, segment tables, raw plane (device)
// One warp per tile, lane l = row l of the tile (tile_n = 32: a lane's symbols are its row, left to right).
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "../../include/anslin.h"
#include "anslin_internal.h"

namespace anslin {
bool normalise_freqs(const uint64_t *cnt, uint32_t *f);   // host.cpp

namespace {

constexpr int kEncWarps = 4;
constexpr int kMaxSeg = 8;   // tile_k <= 1024 weights -> at most 1024 steps = 8 segments of 128

struct EncGeom {
  uint32_t fmt, flags, n_tiles, KT, steps, nseg, seg /*steps per segment*/;
  uint32_t es;            // bytes of one coded symbol's source element along a row: bf16 2, every other format 1
  uint64_t row_bytes;     // bytes of one row of W
  uint32_t raw_tile_bytes;
};

__device__ __forceinline__ const uint8_t *tile_row(const EncGeom &g, const uint8_t *w, uint32_t tile, int lane) {
  const uint32_t grp = tile >> 2, q = tile & 3u, stripe = grp / g.KT, kt = grp % g.KT;
  return w + (uint64_t(stripe) * kTileN + q * 32u + uint32_t(lane)) * g.row_bytes + uint64_t(kt) * g.steps * g.es;
}
__device__ __forceinline__ uint32_t coded_at(const EncGeom &g, const uint8_t *row, int t) {
  if (g.es == 2) return (uint32_t(reinterpret_cast<const uint16_t *>(row)[t]) >> 7) & 0xFFu;
  return row[t];
}
__device__ __forceinline__ uint32_t raw_at(const uint8_t *row, int t) {   // bf16: mantissa << 1 | sign
  const uint32_t v = reinterpret_cast<const uint16_t *>(row)[t];
  return ((v & 0x7Fu) << 1) | (v >> 15);
}
// start state of a lane: L, plus (payload flag) the raw bytes of its last two steps (reading A4)
__device__ __forceinline__ uint32_t start_state(const EncGeom &g, const uint8_t *row) {
  if (!(g.flags & ANSLIN_FLAG_STATE_PAYLOAD)) return kL;
  return kL + (raw_at(row, int(g.steps) - 2) | (raw_at(row, int(g.steps) - 1) << 8));
}
// one encoder step (textbook rANS, P:l.268-279 run backwards): returns true if a word (x & 0xFFFF, before the shift) is emitted
__device__ __forceinline__ bool enc_step(uint32_t &x, uint2 e /* f, start */, uint32_t &word) {
  const bool emit = x >= (e.x << (32 - kProbBits));   // x_max = ((L >> b) << w) * f = f << 20
  word = x & 0xFFFFu;
  if (emit) x >>= kWordBits;
  x = (x / e.x) * kM + (x % e.x) + e.y;
  return emit;
}
__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  return v;
}
__device__ __forceinline__ uint32_t warp_min(uint32_t v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v = min(v, __shfl_xor_sync(0xffffffffu, v, d));
  return v;
}
__device__ __forceinline__ uint32_t warp_max(uint32_t v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, d));
  return v;
}

// status[0] = 1 if some tile does not fit the segment tables, status[1] = largest staged segment in bytes
__global__ void __launch_bounds__(kEncWarps * 32) enc_count_kernel(EncGeom g, const uint8_t *__restrict__ w, const uint2 *__restrict__ tab,
                                                                   uint16_t *__restrict__ counts, uint32_t *__restrict__ sizes,
                                                                   uint32_t *__restrict__ status) {
  __shared__ uint2 stab[256];
  for (int i = threadIdx.x; i < 256; i += blockDim.x) stab[i] = tab[i];
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (uint32_t tile = blockIdx.x * kEncWarps + warp; tile < g.n_tiles; tile += gridDim.x * kEncWarps) {
    const uint8_t *row = tile_row(g, w, tile, lane);
    uint32_t x = start_state(g, row), words = 0, seg_max = 0;
    bool bad = false;
    for (int sg = int(g.nseg) - 1; sg >= 0; --sg) {
      uint32_t c = 0, word;
      for (int t = (sg + 1) * int(g.seg) - 1; t >= sg * int(g.seg); --t) c += enc_step(x, stab[coded_at(g, row, t)], word) ? 1u : 0u;
      counts[(size_t(tile) * g.nseg + sg) * 32 + lane] = uint16_t(c);
      const uint32_t pair = c + __shfl_xor_sync(0xffffffffu, c, 1), total = warp_sum(c);
      bad |= warp_max(pair) - warp_min(pair) > 255u || total > 0xFFFFu;
      words += total;
      seg_max = max(seg_max, ((15u + 2u * total + 15u) & ~15u) + 16u);
    }
    if (lane == 0) {
      sizes[tile] = (4u * kLanes + uint32_t(kSegTableBytes) * g.nseg + 2u * words + 15u) >> 4;
      atomicMax(status + 1, seg_max);
      if (bad) atomicExch(status, 1u);
    }
  }
}

__global__ void __launch_bounds__(kEncWarps * 32) enc_write_kernel(EncGeom g, const uint8_t *__restrict__ w, const uint2 *__restrict__ tab,
                                                                   const uint16_t *__restrict__ counts, const uint32_t *__restrict__ offs,
                                                                   uint8_t *__restrict__ records, uint8_t *__restrict__ raw_plane) {
  __shared__ uint2 stab[256];
  for (int i = threadIdx.x; i < 256; i += blockDim.x) stab[i] = tab[i];
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (uint32_t tile = blockIdx.x * kEncWarps + warp; tile < g.n_tiles; tile += gridDim.x * kEncWarps) {
    const uint8_t *row = tile_row(g, w, tile, lane);
    uint8_t *rec = records + size_t(offs[tile]) * 16;
    // segment tables, and this lane's first write position in every segment
    uint32_t cur[kMaxSeg];
    uint32_t seg_base = 4u * kLanes + uint32_t(kSegTableBytes) * g.nseg;   // byte offset of the segment's words in the record
#pragma unroll
    for (int sg = 0; sg < kMaxSeg; ++sg) {
      cur[sg] = 0;
      if (sg < int(g.nseg)) {
        const uint32_t c = counts[(size_t(tile) * g.nseg + sg) * 32 + lane];
        const uint32_t pair = c + __shfl_xor_sync(0xffffffffu, c, 1), total = warp_sum(c), base = warp_min(pair);
        uint32_t end = (lane & 1) ? 0u : pair;   // inclusive sum over regions 0..p, seen by both lanes of region p
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const uint32_t o = __shfl_up_sync(0xffffffffu, end, d);
          if (lane >= d) end += o;
        }
        const uint32_t start = end - pair;
        // the encoder emits in reverse read order: lane 2p (read ascending from the region start) writes downwards
        // from start + c - 1, lane 2p+1 (read descending from the region end) writes upwards from end - c
        cur[sg] = seg_base + 2u * ((lane & 1) ? end - c : start + c - 1u);
        uint8_t *te = rec + 4 * kLanes + kSegTableBytes * sg;
        if (lane == 0) {
          reinterpret_cast<uint16_t *>(te)[0] = uint16_t(base);
          reinterpret_cast<uint16_t *>(te)[1] = uint16_t(total);
        }
        if (!(lane & 1)) te[4 + (lane >> 1)] = uint8_t(pair - base);
        seg_base += 2u * total;
      }
    }
    const int dir = (lane & 1) ? 2 : -2;
    uint32_t x = start_state(g, row);
#pragma unroll
    for (int sg = kMaxSeg - 1; sg >= 0; --sg) {
      if (sg < int(g.nseg)) {
        uint32_t at = cur[sg], word;
        for (int t = (sg + 1) * int(g.seg) - 1; t >= sg * int(g.seg); --t) {
          if (enc_step(x, stab[coded_at(g, row, t)], word)) {
            *reinterpret_cast<uint16_t *>(rec + at) = uint16_t(word);
            at += uint32_t(dir);
          }
        }
      }
    }
    reinterpret_cast<uint32_t *>(rec)[lane] = x;   // the encoder's final state is the decoder's start state
    if (g.es == 2) {   // bf16 raw plane: 16-step vectors, vector v of lane l at v*512 + l*16
      uint8_t *rp = raw_plane + size_t(tile) * g.raw_tile_bytes;
      const int V = int(g.steps) / 16;
      const bool payload = g.flags & ANSLIN_FLAG_STATE_PAYLOAD;
      for (int v = 0; v < V; ++v) {
        uint32_t r[4] = {0, 0, 0, 0};
#pragma unroll
        for (int i = 0; i < 16; ++i) r[i >> 2] |= raw_at(row, v * 16 + i) << (8 * (i & 3));
        if (!payload || v < V - 1) {
          *reinterpret_cast<uint4 *>(rp + size_t(v) * 512 + lane * 16) = make_uint4(r[0], r[1], r[2], r[3]);
        } else {   // last vector: bytes 14, 15 ride in the start state; the rest as 7 sub-rows of 32 x 2 bytes
#pragma unroll
          for (int h = 0; h < 7; ++h)
            *reinterpret_cast<uint16_t *>(rp + size_t(v) * 512 + h * 64 + lane * 2) = uint16_t(r[h >> 1] >> (16 * (h & 1)));
        }
      }
    }
  }
}

struct EncLayout {   // workspace carve-up
  size_t tab, status, hist, sizes, counts, total;
};
EncLayout enc_layout(uint32_t n_tiles, uint32_t nseg) {
  EncLayout l;
  l.tab = 0;                       // 256 x uint2
  l.status = 2048;                 // 2 x u32
  l.hist = 2048 + 64;              // 2 x 256 x u64
  l.sizes = align16(l.hist + 4096);
  l.counts = align16(l.sizes + 4 * size_t(n_tiles + 1));
  l.total = align16(l.counts + size_t(n_tiles) * nseg * 64);
  return l;
}

bool enc_geometry(const anslin_desc *d, EncGeom *g, uint32_t *n_out, uint32_t *k_in, uint32_t *group) {
  if (!d || d->format > kFormatMax) return false;
  const uint32_t tile_k = d->tile_k ? d->tile_k : 256u, tile_n = d->tile_n;
  if (tile_n != 32 || !(d->flags & ANSLIN_FLAG_LANE_STREAMS)) return false;          // the layout this encoder writes
  if (d->flags & ~(ANSLIN_FLAG_STATE_PAYLOAD | ANSLIN_FLAG_LANE_STREAMS)) return false;
  if ((d->flags & ANSLIN_FLAG_STATE_PAYLOAD) && d->format != ANSLIN_FMT_BF16) return false;
  if (d->n_out == 0 || d->k_in == 0 || d->n_out % kTileN || d->k_in % tile_k || tile_k % 64 || tile_k > 1024) return false;
  if (d->format == ANSLIN_FMT_INT4_AWQ && (d->group_size == 0 || d->group_size % 16 || d->k_in % d->group_size)) return false;
  const uint32_t wps = uint32_t(weights_per_symbol(d->format));
  g->fmt = d->format; g->flags = d->flags;
  g->steps = tile_k / wps;
  g->seg = uint32_t(seg_steps_of(d->format));
  if (g->steps % g->seg) return false;
  g->nseg = g->steps / g->seg;
  if (g->nseg > uint32_t(kMaxSeg) || d->format == ANSLIN_FMT_BF16_PAIR4) return false;   // (the pair variant is host-encoded only)
  g->KT = d->k_in / tile_k;
  g->n_tiles = (d->n_out / kTileN) * g->KT * 4u;
  g->es = d->format == ANSLIN_FMT_BF16 ? 2u : 1u;
  g->row_bytes = d->format == ANSLIN_FMT_BF16 ? uint64_t(d->k_in) * 2 : uint64_t(d->k_in) / wps;
  g->raw_tile_bytes = d->format == ANSLIN_FMT_BF16 ? uint32_t(raw_tile_bytes(32, tile_k, d->flags)) : 0u;
  *n_out = d->n_out; *k_in = d->k_in; *group = d->group_size;
  return true;
}

}  // namespace
}  // namespace anslin

extern "C" int anslin_histogram(uint32_t format, const void *w_dev, uint64_t n_elems, void *counts_dev, void *stream);

extern "C" size_t anslin_encode_device_workspace_bytes(const anslin_desc *desc) {
  using namespace anslin;
  EncGeom g;
  uint32_t n_out, k_in, group;
  if (!enc_geometry(desc, &g, &n_out, &k_in, &group)) return 0;
  return enc_layout(g.n_tiles, g.nseg).total;
}

extern "C" size_t anslin_encode_device_head_bytes(const anslin_desc *desc) {
  using namespace anslin;
  EncGeom g;
  uint32_t n_out, k_in, group;
  if (!enc_geometry(desc, &g, &n_out, &k_in, &group)) return 0;
  return align16(align16(size_t(kHeaderBytes) + 512) + 4 * size_t(g.n_tiles + 1));
}

extern "C" int anslin_encode_device(const anslin_desc *desc, const void *w_dev, const void *scales_host, const void *zeros_host,
                                    void *container_dev, size_t capacity, void *head_host, size_t head_capacity, void *workspace_dev,
                                    size_t workspace_bytes, size_t *bytes_out, void *stream) {
  using namespace anslin;
  if (!desc || !w_dev || !container_dev || !head_host || !workspace_dev || !bytes_out) return ANSLIN_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(w_dev) | reinterpret_cast<uintptr_t>(container_dev) | reinterpret_cast<uintptr_t>(workspace_dev)) & 15)
    return ANSLIN_ERR_INVALID_ARG;
  EncGeom g;
  uint32_t n_out, k_in, group;
  if (!enc_geometry(desc, &g, &n_out, &k_in, &group)) return ANSLIN_ERR_UNSUPPORTED;
  if (g.fmt == ANSLIN_FMT_INT8 && !scales_host) return ANSLIN_ERR_INVALID_ARG;
  if (g.fmt == ANSLIN_FMT_INT4_AWQ && (!scales_host || !zeros_host)) return ANSLIN_ERR_INVALID_ARG;
  const EncLayout L = enc_layout(g.n_tiles, g.nseg);
  if (workspace_bytes < L.total) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint8_t *ws = static_cast<uint8_t *>(workspace_dev), *out = static_cast<uint8_t *>(container_dev);
  const uint8_t *w = static_cast<const uint8_t *>(w_dev);

  // 1-2. histogram of the coded symbols -> 12-bit table
  const uint64_t n_elems = g.fmt == ANSLIN_FMT_BF16 ? uint64_t(n_out) * k_in : uint64_t(n_out) * g.row_bytes;
  int rc = anslin_histogram(g.fmt, w_dev, n_elems, ws + L.hist, st);
  if (rc != ANSLIN_OK) return rc;
  uint64_t cnt[256];
  if (cudaMemcpyAsync(cnt, ws + L.hist, sizeof(cnt), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess)
    return ANSLIN_ERR_CUDA;
  uint32_t f[256];
  if (!normalise_freqs(cnt, f)) return ANSLIN_ERR_INVALID_ARG;
  uint2 tab[256];
  uint32_t run = 0;
  for (int s = 0; s < 256; ++s) { tab[s] = make_uint2(f[s] ? f[s] : 1u, run); run += f[s]; }   // dead symbols never occur: f = 1 avoids x / 0
  const uint32_t zero2[2] = {0, 0};
  if (cudaMemcpyAsync(ws + L.tab, tab, sizeof(tab), cudaMemcpyHostToDevice, st) != cudaSuccess ||
      cudaMemcpyAsync(ws + L.status, zero2, sizeof(zero2), cudaMemcpyHostToDevice, st) != cudaSuccess)
    return ANSLIN_ERR_CUDA;

  // 3. word counts -> record sizes
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0)
    return ANSLIN_ERR_CUDA;
  const uint32_t grid = std::min<uint32_t>((g.n_tiles + kEncWarps - 1) / kEncWarps, uint32_t(sms) * 8u);
  enc_count_kernel<<<grid, kEncWarps * 32, 0, st>>>(g, w, reinterpret_cast<const uint2 *>(ws + L.tab), reinterpret_cast<uint16_t *>(ws + L.counts),
                                                    reinterpret_cast<uint32_t *>(ws + L.sizes), reinterpret_cast<uint32_t *>(ws + L.status));
  std::vector<uint32_t> sizes(g.n_tiles + 1);
  uint32_t status[2];
  if (cudaMemcpyAsync(sizes.data(), ws + L.sizes, 4 * size_t(g.n_tiles), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaMemcpyAsync(status, ws + L.status, sizeof(status), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess)
    return ANSLIN_ERR_CUDA;
  if (status[0]) return ANSLIN_ERR_UNSUPPORTED;   // a tile's region sizes do not fit the segment tables (the host encoder falls back to interleaved words)

  // 4. offsets and section layout (identical to anslin_encode_host's)
  uint64_t pos = 0;
  for (uint32_t t = 0; t < g.n_tiles; ++t) { const uint32_t sz = sizes[t]; sizes[t] = uint32_t(pos); pos += sz; }
  sizes[g.n_tiles] = uint32_t(pos);
  if (pos > 0xFFFFFFFFull) return ANSLIN_ERR_UNSUPPORTED;
  const uint64_t rec_total = pos * 16;
  Header h;
  memset(&h, 0, sizeof(h));
  h.off_freq = kHeaderBytes;
  h.off_offsets = align16(h.off_freq + 512);
  h.off_records = align16(h.off_offsets + 4 * size_t(g.n_tiles + 1));
  const uint64_t raw_total = uint64_t(g.raw_tile_bytes) * g.n_tiles;
  const uint64_t sb = g.fmt == ANSLIN_FMT_INT8 ? uint64_t(2) * n_out : g.fmt == ANSLIN_FMT_INT4_AWQ ? uint64_t(4) * n_out * (k_in / group) : 0;
  h.off_raw = raw_total ? align16(h.off_records + rec_total) : 0;
  const uint64_t after_raw = raw_total ? h.off_raw + raw_total : h.off_records + rec_total;
  h.off_scales = sb ? align16(after_raw) : 0;
  h.total_bytes = align16(sb ? h.off_scales + sb : after_raw);
  h.total_bytes = std::max<uint64_t>(h.total_bytes, align16(h.off_records + rec_total + kTailBytes));
  *bytes_out = h.total_bytes;
  if (h.total_bytes > capacity) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  if (head_capacity < h.off_records) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  h.magic = kMagic; h.version = kVersion; h.format = g.fmt; h.n_out = n_out; h.k_in = k_in; h.tile_n = 32;
  h.tile_k = desc->tile_k ? desc->tile_k : 256u; h.streams = kLanes; h.prob_bits = kProbBits; h.word_bits = kWordBits;
  h.state_lo_log2 = kStateLoLog2; h.group_size = group; h.flags = g.flags; h.n_tiles = g.n_tiles;
  h.w_scale = is_fp8_path(g.fmt) ? desc->w_scale : 1.0f;
  h.max_seg_bytes = status[1];
  uint8_t *head = static_cast<uint8_t *>(head_host);
  memset(head, 0, h.off_records);
  memcpy(head, &h, sizeof(h));
  for (int s = 0; s < 256; ++s) reinterpret_cast<uint16_t *>(head + h.off_freq)[s] = uint16_t(f[s]);
  memcpy(head + h.off_offsets, sizes.data(), 4 * size_t(g.n_tiles + 1));
  if (cudaMemsetAsync(out, 0, h.total_bytes, st) != cudaSuccess ||
      cudaMemcpyAsync(out, head, h.off_records, cudaMemcpyHostToDevice, st) != cudaSuccess)
    return ANSLIN_ERR_CUDA;
  std::vector<uint16_t> side;
  if (g.fmt == ANSLIN_FMT_INT8) {
    if (cudaMemcpyAsync(out + h.off_scales, scales_host, sb, cudaMemcpyHostToDevice, st) != cudaSuccess) return ANSLIN_ERR_CUDA;
  } else if (g.fmt == ANSLIN_FMT_INT4_AWQ) {   // (scale, zero) fp16 pairs, [group][n_out]
    const uint16_t *s = static_cast<const uint16_t *>(scales_host), *z = static_cast<const uint16_t *>(zeros_host);
    const size_t groups = k_in / group;
    side.resize(size_t(2) * groups * n_out);
    for (size_t gi = 0; gi < groups; ++gi)
      for (size_t n = 0; n < n_out; ++n) {
        side[(gi * n_out + n) * 2 + 0] = s[n * groups + gi];
        side[(gi * n_out + n) * 2 + 1] = z[n * groups + gi];
      }
    if (cudaMemcpyAsync(out + h.off_scales, side.data(), sb, cudaMemcpyHostToDevice, st) != cudaSuccess) return ANSLIN_ERR_CUDA;
  }

  // 5. write the records (and the bf16 raw plane)
  enc_write_kernel<<<grid, kEncWarps * 32, 0, st>>>(g, w, reinterpret_cast<const uint2 *>(ws + L.tab), reinterpret_cast<const uint16_t *>(ws + L.counts),
                                                    reinterpret_cast<const uint32_t *>(out + h.off_offsets), out + h.off_records,
                                                    raw_total ? out + h.off_raw : nullptr);
  if (cudaGetLastError() != cudaSuccess) return ANSLIN_ERR_CUDA;
  // `side` and the pageable copies above must outlive their transfers: this offline call ends synchronised
  return cudaStreamSynchronize(st) == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}
