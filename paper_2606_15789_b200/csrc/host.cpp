// libanslin host side: offline encoder / tile packer (anslin_encode_host), container validation
// (anslin_open) and small helpers.  Plain C++17, no CUDA.  Independent of oracle/.
//
// Paper passages: P:l.165-169 §V-B (offline stage), P:l.149 §IV-A (tile-partitioned bitstreams,
// shared codebook, tile index table), P:l.192 (R interleaved substreams), Eq.3 P:l.440.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <new>
#include <thread>
#include <vector>

#include "anslin_internal.h"

using namespace anslin;

namespace {

struct Geometry {
  uint32_t fmt, n_out, k_in, tile_n, tile_k, flags, group;
  int spc, wps, sym_cols /*symbols per tile row*/, units, steps, KT, stripes, Q /*tiles per (stripe, k-tile) group*/, rb /*tile_n / 32*/;
  size_t n_tiles, row_syms /*symbols per matrix row*/;
  uint8_t code_of[256];   // bf16 pair variant: exponent byte -> 4-bit code (15 = escape)
  uint8_t codes[16];      //                    code -> exponent byte (the container's code table)
};

bool make_geometry(const anslin_desc *d, Geometry *g) {
  if (!d || d->format > kFormatMax) return false;
  g->fmt = d->format;
  g->n_out = d->n_out;
  g->k_in = d->k_in;
  g->tile_k = d->tile_k ? d->tile_k : default_tile_k(d->format);
  g->tile_n = d->tile_n ? d->tile_n : uint32_t(kTileN);
  if (g->tile_n != 32 && g->tile_n != uint32_t(kTileN)) return false;
  g->flags = d->flags;
  g->group = d->group_size;
  g->spc = spc_of(g->fmt);
  g->wps = weights_per_symbol(g->fmt);
  if (g->n_out == 0 || g->k_in == 0 || g->n_out % kTileN || g->k_in % g->tile_k) return false;
  if (g->tile_k % unit_k_of(g->fmt) || g->tile_k % 64 || g->tile_k > 1024) return false;
  if ((g->flags & ~(ANSLIN_FLAG_STATE_PAYLOAD | ANSLIN_FLAG_LANE_STREAMS)) != 0) return false;
  if ((g->flags & ANSLIN_FLAG_STATE_PAYLOAD) && !is_bf16_like(g->fmt)) return false;
  if (g->fmt == ANSLIN_FMT_BF16_PAIR4 && (!(g->flags & ANSLIN_FLAG_LANE_STREAMS) || g->tile_n != 32)) return false;
  if (g->fmt == ANSLIN_FMT_INT4_AWQ && (g->group == 0 || g->group % 16 || g->k_in % g->group)) return false;
  g->sym_cols = int(g->tile_k) / g->wps;
  g->units = g->sym_cols / (2 * g->spc);
  g->rb = int(g->tile_n) / 32;
  g->Q = kTileN / int(g->tile_n);
  g->steps = g->units * 2 * g->rb * g->spc;
  g->KT = int(g->k_in / g->tile_k);
  g->stripes = int(g->n_out / kTileN);
  g->n_tiles = size_t(g->KT) * g->stripes * g->Q;
  if ((g->flags & ANSLIN_FLAG_LANE_STREAMS) && (g->tile_n != 32 || g->steps % seg_steps_of(g->fmt))) return false;
  g->row_syms = g->k_in / g->wps;
  return true;
}

size_t side_bytes(const Geometry &g) {
  if (g.fmt == ANSLIN_FMT_INT8) return size_t(2) * g.n_out;
  if (g.fmt == ANSLIN_FMT_INT4_AWQ) return size_t(4) * g.n_out * (g.k_in / g.group);
  return 0;
}

// Coded symbol / raw byte of the weight element at (row, symbol column) of W.
inline uint8_t coded_symbol(const Geometry &g, const void *w, size_t row, size_t col) {
  if (g.fmt == ANSLIN_FMT_BF16) return uint8_t(reinterpret_cast<const uint16_t *>(w)[row * g.k_in + col] >> 7);
  if (g.fmt == ANSLIN_FMT_BF16_PAIR4) {   // col counts weight PAIRS
    const uint16_t *p = reinterpret_cast<const uint16_t *>(w) + row * g.k_in + 2 * col;
    return uint8_t(g.code_of[uint8_t(p[0] >> 7)] | (g.code_of[uint8_t(p[1] >> 7)] << 4));
  }
  return reinterpret_cast<const uint8_t *>(w)[row * g.row_syms + col];
}
inline uint8_t raw_byte(const Geometry &g, const void *w, size_t row, size_t col) {
  uint16_t v = reinterpret_cast<const uint16_t *>(w)[row * g.k_in + col];
  return uint8_t(((v & 0x7F) << 1) | (v >> 15));
}

// 12-bit frequency normalisation: every live symbol keeps f >= 1, sum f = 4096, and units are
// handed out / taken back where they change the coded size least (A10).
bool normalise(const uint64_t *cnt, uint32_t *f) {
  uint64_t n = 0;
  int live = 0, only = -1;
  for (int s = 0; s < 256; ++s) {
    n += cnt[s];
    if (cnt[s]) { ++live; only = s; }
  }
  if (!live) return false;
  std::fill(f, f + 256, 0u);
  if (live == 1) {  // DESIGN.md A11: f must fit 12 bits
    f[only] = kM - 1;
    f[(only + 1) & 255] = 1;
    return true;
  }
  int64_t sum = 0;
  for (int s = 0; s < 256; ++s)
    if (cnt[s]) {
      uint64_t q = uint64_t((long double)cnt[s] * kM / (long double)n);
      f[s] = uint32_t(std::max<uint64_t>(1, q));
      sum += f[s];
    }
  while (sum != int64_t(kM)) {
    int best = -1;
    double bestv = 0;
    for (int s = 0; s < 256; ++s) {
      if (!cnt[s]) continue;
      if (sum < int64_t(kM)) {
        double v = double(cnt[s]) * std::log2(double(f[s] + 1) / double(f[s]));
        if (best < 0 || v > bestv) { best = s; bestv = v; }
      } else if (f[s] > 1) {
        double v = double(cnt[s]) * std::log2(double(f[s]) / double(f[s] - 1));
        if (best < 0 || v < bestv) { best = s; bestv = v; }
      }
    }
    if (sum < int64_t(kM)) { ++f[best]; ++sum; } else { --f[best]; --sum; }
  }
  return true;
}

// One tile -> record bytes (32 states + words in decoder read order + pad) and raw plane bytes.
// Returns false if the lane-stream layout cannot represent the tile.  *seg_bytes_out: staged bytes of its largest segment.
bool encode_tile(const Geometry &g, const void *w, size_t tile, const uint32_t *f, const uint32_t *c,
                 std::vector<uint8_t> &rec, uint8_t *raw_out, uint64_t *n_words_out, uint32_t *seg_bytes_out) {
  const int steps = g.steps, spc = g.spc, G = 2 * g.rb;
  const size_t grp = tile / g.Q, q = tile % g.Q, stripe = grp / g.KT, kt = grp % g.KT;
  const size_t row0 = stripe * kTileN + q * g.tile_n, col0 = kt * g.sym_cols;
  const bool pair = g.fmt == ANSLIN_FMT_BF16_PAIR4;
  std::vector<uint8_t> sym(size_t(steps) * kLanes), raw;
  if (g.fmt == ANSLIN_FMT_BF16) raw.resize(sym.size());
  if (pair) {   // one raw byte per WEIGHT: raw[k * 32 + lane], lane = row (32-row tiles)
    raw.resize(size_t(g.tile_k) * kLanes);
    for (size_t k = 0; k < g.tile_k; ++k)
      for (int lane = 0; lane < kLanes; ++lane) raw[k * kLanes + lane] = raw_byte(g, w, row0 + lane, size_t(kt) * g.tile_k + k);
  }
  const size_t raw_steps = pair ? g.tile_k : size_t(steps);   // entries per lane in raw[]
  for (int u = 0; u < g.units; ++u)
    for (int gq = 0; gq < G; ++gq)
      for (int lane = 0; lane < kLanes; ++lane) {
        size_t row = row0 + size_t((gq % g.rb) * 32 + lane), col = col0 + size_t(u) * 2 * spc + size_t(gq / g.rb) * spc;
        for (int e = 0; e < spc; ++e) {
          size_t t = size_t(u * G + gq) * spc + e;
          sym[t * kLanes + lane] = coded_symbol(g, w, row, col + e);
          if (!raw.empty() && !pair) raw[t * kLanes + lane] = raw_byte(g, w, row, col + e);
        }
      }
  uint32_t x[kLanes];
  const bool payload = g.flags & ANSLIN_FLAG_STATE_PAYLOAD;
  for (int lane = 0; lane < kLanes; ++lane) {
    x[lane] = kL;
    if (payload)
      x[lane] += uint32_t(raw[(raw_steps - 2) * kLanes + lane]) | (uint32_t(raw[(raw_steps - 1) * kLanes + lane]) << 8);
  }
  // Words are produced back to front so that the buffer ends up in decoder read order
  // (step ascending, renormalising lanes ascending) without a reversal pass.
  const bool lane_streams = g.flags & ANSLIN_FLAG_LANE_STREAMS;
  const int seg = seg_steps_of(g.fmt);
  const int S = lane_streams ? steps / seg : 0;
  std::vector<uint16_t> words(lane_streams ? 0 : sym.size() + 8);
  std::vector<std::vector<uint16_t>> lw(size_t(S) * kLanes);   // lane streams: words of (segment, lane), filled back to front
  size_t wp = words.size();
  for (int t = steps; t-- > 0;)
    for (int lane = kLanes; lane-- > 0;) {
      const uint8_t s = sym[size_t(t) * kLanes + lane];
      const uint32_t fs = f[s];
      uint32_t xv = x[lane];
      if (pair && (t & 3) == 3) {
        // escape literals of the 4-step chunk: read after the chunk's last renormalisation in weight order, so (this
        // buffer is filled back to front) pushed first, last weight first
        const uint16_t *pw = reinterpret_cast<const uint16_t *>(w) + (row0 + lane) * size_t(g.k_in) + size_t(kt) * g.tile_k;
        for (int tt = t; tt > t - 4; --tt) {
          const uint8_t sc = sym[size_t(tt) * kLanes + lane];
          if ((sc >> 4) == 15) lw[size_t(t / seg) * kLanes + lane].push_back(uint16_t(uint8_t(pw[2 * tt + 1] >> 7)));
          if ((sc & 15) == 15) lw[size_t(t / seg) * kLanes + lane].push_back(uint16_t(uint8_t(pw[2 * tt] >> 7)));
        }
      }
      if (uint64_t(xv) >= (uint64_t(fs) << (kStateLoLog2 - kProbBits + kWordBits))) {
        // the decoder reads this word right after decoding step t
        if (lane_streams) lw[size_t(t / seg) * kLanes + lane].push_back(uint16_t(xv));
        else words[--wp] = uint16_t(xv);
        xv >>= kWordBits;
      }
      x[lane] = ((xv / fs) << kProbBits) + (xv % fs) + c[s];
    }
  *seg_bytes_out = 0;
  if (lane_streams) {
    // record = states | per segment {u16 base, u16 total, 16 x u8 delta} | per segment 16 regions: lane 2p ascending,
    // lane 2p+1 descending from the region end (lw holds every lane's words in REVERSE read order already)
    size_t nw = 0;
    for (auto &v : lw) nw += v.size();
    rec.assign(align16(4 * kLanes + size_t(kSegTableBytes) * S + 2 * nw), 0);
    std::memcpy(rec.data(), x, 4 * kLanes);
    uint8_t *tabp = rec.data() + 4 * kLanes;
    uint16_t *wout = reinterpret_cast<uint16_t *>(tabp + size_t(kSegTableBytes) * S);
    for (int sg = 0; sg < S; ++sg) {
      size_t sizes[kLanes / 2], base = ~size_t(0), total = 0;
      for (int p = 0; p < kLanes / 2; ++p) {
        sizes[p] = lw[size_t(sg) * kLanes + 2 * p].size() + lw[size_t(sg) * kLanes + 2 * p + 1].size();
        base = std::min(base, sizes[p]);
        total += sizes[p];
      }
      if (total > 0xFFFF) return false;
      uint16_t hdr[2] = {uint16_t(base), uint16_t(total)};
      std::memcpy(tabp + size_t(kSegTableBytes) * sg, hdr, 4);
      for (int p = 0; p < kLanes / 2; ++p) {
        if (sizes[p] - base > 255) return false;
        tabp[size_t(kSegTableBytes) * sg + 4 + p] = uint8_t(sizes[p] - base);
        const auto &ev = lw[size_t(sg) * kLanes + 2 * p], &od = lw[size_t(sg) * kLanes + 2 * p + 1];
        for (size_t i = ev.size(); i-- > 0;) *wout++ = ev[i];       // read order ascending
        for (size_t i = 0; i < od.size(); ++i) *wout++ = od[i];     // reverse read order: lane 2p+1 walks down from the end
      }
      *seg_bytes_out = std::max<uint32_t>(*seg_bytes_out, uint32_t(align16(15 + 2 * total) + 16));
    }
    *n_words_out = nw;
  } else {
    const size_t nw = words.size() - wp;
    rec.assign(align16(4 * kLanes + 2 * nw), 0);
    std::memcpy(rec.data(), x, 4 * kLanes);
    std::memcpy(rec.data() + 4 * kLanes, words.data() + wp, 2 * nw);
    *n_words_out = nw;
  }
  if (raw_out) {
    const int V = int(raw_steps / 16);
    for (int v = 0; v < V; ++v) {
      const bool last = payload && v == V - 1;
      for (int lane = 0; lane < kLanes; ++lane)
        for (int p = 0; p < (last ? 14 : 16); ++p) {
          uint8_t b = raw[size_t(v * 16 + p) * kLanes + lane];
          if (!last) raw_out[size_t(v) * 512 + lane * 16 + p] = b;
          else raw_out[size_t(v) * 512 + (p >> 1) * 64 + lane * 2 + (p & 1)] = b;
        }
    }
  }
  return true;
}

int encode_with(Geometry g, const anslin_desc *desc, const void *w_host, const void *scales_host, const void *zeros_host,
                void *container_out, size_t capacity, size_t *bytes_out, anslin_stats *st);

}  // namespace

namespace anslin {
// the encoder's table normalisation, shared with the device-side encoder (encode_gpu.cu)
bool normalise_freqs(const uint64_t *cnt, uint32_t *f) { return normalise(cnt, f); }
}  // namespace anslin

extern "C" {

size_t anslin_encode_bound(const anslin_desc *desc) {
  Geometry g;
  if (!make_geometry(desc, &g)) return 0;
  const size_t tile_syms = size_t(g.steps) * kLanes;
  // every symbol costs at most 12 bits + one flush word per lane; round generously
  // pair variant: a step may also carry two literal words
  const size_t words_max = g.fmt == ANSLIN_FMT_BF16_PAIR4 ? tile_syms * 3 : tile_syms * 3 / 4;
  const size_t rec = align16(4 * kLanes + 2 * (words_max + 2 * kLanes + 8)) + align16(size_t(kSegTableBytes) * (g.steps / seg_steps_of(g.fmt) + 1));
  size_t total = kHeaderBytes + 512 + align16(4 * (g.n_tiles + 1)) + g.n_tiles * rec + 64;
  if (is_bf16_like(g.fmt)) total += g.n_tiles * raw_tile_bytes(g.tile_n, g.tile_k, 0) + 16 + 32;
  return total + align16(side_bytes(g)) + 16 + kTailBytes;
}

int anslin_encode_host(const anslin_desc *desc, const void *w_host, const void *scales_host, const void *zeros_host,
                       void *container_out, size_t capacity, size_t *bytes_out, anslin_stats *st) {
  if (!desc || !w_host || !container_out || !bytes_out) return ANSLIN_ERR_INVALID_ARG;
  if (desc->format > kFormatMax) return ANSLIN_ERR_UNSUPPORTED;
  Geometry g;
  if (!make_geometry(desc, &g)) return ANSLIN_ERR_UNSUPPORTED;
  return encode_with(g, desc, w_host, scales_host, zeros_host, container_out, capacity, bytes_out, st);
}

}  // extern "C"

namespace {
int encode_with(Geometry g, const anslin_desc *desc, const void *w_host, const void *scales_host, const void *zeros_host,
                void *container_out, size_t capacity, size_t *bytes_out, anslin_stats *st) {
  if (g.fmt == ANSLIN_FMT_INT8 && !scales_host) return ANSLIN_ERR_INVALID_ARG;
  if (g.fmt == ANSLIN_FMT_INT4_AWQ && (!scales_host || !zeros_host)) return ANSLIN_ERR_INVALID_ARG;

  unsigned nthr = std::max(1u, std::min(32u, std::thread::hardware_concurrency()));
  if (g.n_tiles < 64) nthr = 1;

  if (g.fmt == ANSLIN_FMT_BF16_PAIR4) {
    // code table: the 15 most frequent exponent bytes, descending count, ties by smaller exponent; code 15 = escape
    std::vector<uint64_t> ce(256, 0);
    const uint16_t *p = static_cast<const uint16_t *>(w_host);
    for (size_t i = 0, n = size_t(g.n_out) * g.k_in; i < n; ++i) ++ce[uint8_t(p[i] >> 7)];
    int order[256];
    for (int s = 0; s < 256; ++s) order[s] = s;
    std::stable_sort(order, order + 256, [&](int a, int b) { return ce[a] > ce[b]; });
    std::memset(g.code_of, 15, sizeof(g.code_of));
    std::memset(g.codes, 0, sizeof(g.codes));
    for (int i = 0; i < 15; ++i) { g.codes[i] = uint8_t(order[i]); g.code_of[order[i]] = uint8_t(i); }
  }

  // P:l.167: statistics aggregated over the whole matrix -> one shared codebook.
  std::vector<std::vector<uint64_t>> hist(nthr, std::vector<uint64_t>(512, 0));
  {
    std::vector<std::thread> th;
    for (unsigned i = 0; i < nthr; ++i)
      th.emplace_back([&, i] {
        size_t r0 = size_t(g.n_out) * i / nthr, r1 = size_t(g.n_out) * (i + 1) / nthr;
        uint64_t *hc = hist[i].data(), *hr = hc + 256;
        for (size_t r = r0; r < r1; ++r)
          for (size_t c = 0; c < g.row_syms; ++c) {
            ++hc[coded_symbol(g, w_host, r, c)];
            if (g.fmt == ANSLIN_FMT_BF16) ++hr[raw_byte(g, w_host, r, c)];
            if (g.fmt == ANSLIN_FMT_BF16_PAIR4) { ++hr[raw_byte(g, w_host, r, 2 * c)]; ++hr[raw_byte(g, w_host, r, 2 * c + 1)]; }
          }
      });
    for (auto &t : th) t.join();
  }
  uint64_t cnt[256] = {0}, cnt_raw[256] = {0};
  for (auto &h : hist)
    for (int s = 0; s < 256; ++s) { cnt[s] += h[s]; cnt_raw[s] += h[256 + s]; }
  uint32_t f[256], c[256];
  if (!normalise(cnt, f)) return ANSLIN_ERR_INVALID_ARG;
  for (uint32_t s = 0, acc = 0; s < 256; ++s) { c[s] = acc; acc += f[s]; }

  // Encode tiles in parallel, then lay the records out in tile order.
  std::vector<std::vector<uint8_t>> recs(g.n_tiles);
  std::vector<uint64_t> nwords(g.n_tiles, 0);
  std::vector<uint32_t> segbytes(g.n_tiles, 0);
  std::atomic<bool> lane_fail(false);
  const size_t rtb = is_bf16_like(g.fmt) ? raw_tile_bytes(g.tile_n, g.tile_k, g.flags) : 0;
  Header h;
  std::memset(&h, 0, sizeof(h));
  h.off_freq = kHeaderBytes;
  h.off_offsets = align16(h.off_freq + 512);
  h.off_records = align16(h.off_offsets + 4 * (g.n_tiles + 1));
  // raw plane position depends on the record sizes; stage raw bytes separately first
  std::vector<uint8_t> raw_all;
  try {
    raw_all.resize(rtb * g.n_tiles);
  } catch (const std::bad_alloc &) { return ANSLIN_ERR_BUFFER_TOO_SMALL; }
  {
    std::atomic<size_t> next(0);
    std::vector<std::thread> th;
    for (unsigned i = 0; i < nthr; ++i)
      th.emplace_back([&] {
        for (;;) {
          size_t t = next.fetch_add(1);
          if (t >= g.n_tiles) break;
          if (!encode_tile(g, w_host, t, f, c, recs[t], rtb ? raw_all.data() + t * rtb : nullptr, &nwords[t], &segbytes[t]))
            lane_fail = true;
        }
      });
    for (auto &t : th) t.join();
  }
  if (lane_fail) {   // a tile does not fit the lane-stream tables: encode the matrix with interleaved words instead
    if (g.fmt == ANSLIN_FMT_BF16_PAIR4) return ANSLIN_ERR_UNSUPPORTED;   // the pair variant has no interleaved layout
    g.flags &= ~ANSLIN_FLAG_LANE_STREAMS;
    return encode_with(g, desc, w_host, scales_host, zeros_host, container_out, capacity, bytes_out, st);
  }
  size_t rec_total = 0;
  for (auto &r : recs) rec_total += r.size();
  const size_t sb = side_bytes(g);
  h.off_raw = rtb ? align16(h.off_records + rec_total) : 0;
  const size_t after_raw = rtb ? h.off_raw + raw_all.size() : h.off_records + rec_total;
  h.off_scales = sb ? align16(after_raw) : 0;
  h.total_bytes = align16(sb ? h.off_scales + sb : after_raw);
  if (g.fmt == ANSLIN_FMT_BF16_PAIR4) {   // 16-byte exponent code table, in the section slot no other format uses
    h.off_zeros = align16(after_raw);
    h.total_bytes = h.off_zeros + 16;
  }
  // tail rule: the decoder's compressed-word ring reads ahead of the record it decodes, so at least
  // kTailBytes readable bytes follow the records section (zero padding if the sections after it are short)
  h.total_bytes = std::max<uint64_t>(h.total_bytes, align16(h.off_records + rec_total + kTailBytes));
  *bytes_out = h.total_bytes;
  if (h.total_bytes > capacity) return ANSLIN_ERR_BUFFER_TOO_SMALL;
  if (rec_total / 16 > 0xFFFFFFFFull) return ANSLIN_ERR_UNSUPPORTED;

  h.magic = kMagic; h.version = kVersion; h.format = g.fmt; h.n_out = g.n_out; h.k_in = g.k_in;
  h.tile_n = g.tile_n; h.tile_k = g.tile_k; h.streams = kLanes; h.prob_bits = kProbBits; h.word_bits = kWordBits;
  h.state_lo_log2 = kStateLoLog2; h.group_size = g.group; h.flags = g.flags; h.n_tiles = uint32_t(g.n_tiles);
  h.w_scale = is_fp8_path(g.fmt) ? desc->w_scale : 1.0f;
  for (uint32_t b : segbytes) h.max_seg_bytes = std::max(h.max_seg_bytes, b);

  uint8_t *out = static_cast<uint8_t *>(container_out);
  std::memset(out, 0, h.total_bytes);
  std::memcpy(out, &h, sizeof(h));
  uint16_t *fq = reinterpret_cast<uint16_t *>(out + h.off_freq);
  for (int s = 0; s < 256; ++s) fq[s] = uint16_t(f[s]);
  uint32_t *offs = reinterpret_cast<uint32_t *>(out + h.off_offsets);
  size_t pos = 0;
  uint64_t pad_bits = 0, payload_bits = 0;
  for (size_t t = 0; t < g.n_tiles; ++t) {
    offs[t] = uint32_t(pos / 16);
    std::memcpy(out + h.off_records + pos, recs[t].data(), recs[t].size());
    pos += recs[t].size();
    payload_bits += 16 * nwords[t];
    pad_bits += 8 * (recs[t].size() - 4 * kLanes - 2 * nwords[t]);   // record padding (+ lane-stream segment tables)
  }
  offs[g.n_tiles] = uint32_t(pos / 16);
  if (rtb) std::memcpy(out + h.off_raw, raw_all.data(), raw_all.size());
  if (g.fmt == ANSLIN_FMT_BF16_PAIR4) std::memcpy(out + h.off_zeros, g.codes, 16);
  if (g.fmt == ANSLIN_FMT_INT8) {
    std::memcpy(out + h.off_scales, scales_host, sb);
  } else if (g.fmt == ANSLIN_FMT_INT4_AWQ) {
    // kernel-friendly side layout: (scale, zero) fp16 pairs, [group][n_out]
    const uint16_t *s = static_cast<const uint16_t *>(scales_host), *z = static_cast<const uint16_t *>(zeros_host);
    uint16_t *o = reinterpret_cast<uint16_t *>(out + h.off_scales);
    const size_t groups = g.k_in / g.group;
    for (size_t gi = 0; gi < groups; ++gi)
      for (size_t n = 0; n < g.n_out; ++n) {
        o[(gi * g.n_out + n) * 2 + 0] = s[n * groups + gi];
        o[(gi * g.n_out + n) * 2 + 1] = z[n * groups + gi];
      }
  }
  if (st) {
    std::memset(st, 0, sizeof(*st));
    st->n_weights = uint64_t(g.n_out) * g.k_in;
    st->payload_bits = payload_bits;
    st->state_bits = 32ull * kLanes * g.n_tiles;
    st->pad_bits = pad_bits;
    st->offset_table_bits = 32ull * (g.n_tiles + 1);
    st->freq_table_bits = 512 * 8;
    st->raw_bits = 8ull * raw_all.size();
    st->side_bits = 8ull * sb;
    st->total_bytes = h.total_bytes;
    auto H = [](const uint64_t *cn) {
      double n = 0, e = 0;
      for (int s = 0; s < 256; ++s) n += double(cn[s]);
      for (int s = 0; s < 256; ++s)
        if (cn[s]) { double p = double(cn[s]) / n; e -= p * std::log2(p); }
      return n > 0 ? e : 0.0;
    };
    st->entropy_bits_per_symbol = H(cnt);
    st->raw_entropy_bits_per_symbol = is_bf16_like(g.fmt) ? H(cnt_raw) : 0.0;
    double n = 0, x = 0;
    for (int s = 0; s < 256; ++s) n += double(cnt[s]);
    for (int s = 0; s < 256; ++s)
      if (cnt[s]) x += double(cnt[s]) / n * std::log2(double(kM) / double(f[s]));
    st->xent_bits_per_symbol = x;
    st->bits_per_weight = 8.0 * double(h.total_bytes - sb) / double(st->n_weights);
  }
  return ANSLIN_OK;
}
}  // namespace

extern "C" {

int anslin_open(const void *container_host, size_t bytes, const void *container_dev, anslin_weight **out) {
  if (!container_host || !out || bytes < size_t(kHeaderBytes)) return ANSLIN_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(container_dev) & 15) return ANSLIN_ERR_INVALID_ARG;
  Header h;
  std::memcpy(&h, container_host, sizeof(h));
  if (h.magic != kMagic || h.version != kVersion) return ANSLIN_ERR_CORRUPT;
  anslin_desc d{h.format, h.n_out, h.k_in, h.tile_k, h.group_size, h.flags, h.w_scale, h.tile_n};
  Geometry g;
  if (h.format > kFormatMax || !make_geometry(&d, &g)) return ANSLIN_ERR_CORRUPT;
  if (h.tile_n != g.tile_n || h.streams != kLanes || h.prob_bits != kProbBits || h.word_bits != kWordBits ||
      h.state_lo_log2 != kStateLoLog2 || h.n_tiles != g.n_tiles)
    return ANSLIN_ERR_CORRUPT;
  const uint64_t T = h.total_bytes;
  auto in = [&](uint64_t off, uint64_t len) { return off % 16 == 0 && off >= kHeaderBytes && off <= T && len <= T - off; };
  if (!in(h.off_freq, 512) || !in(h.off_offsets, 4 * (g.n_tiles + 1)) || !in(h.off_records, 0)) return ANSLIN_ERR_CORRUPT;
  if (bytes < h.off_offsets + 4 * (g.n_tiles + 1)) return ANSLIN_ERR_INVALID_ARG;
  const uint8_t *p = static_cast<const uint8_t *>(container_host);
  const uint16_t *fq = reinterpret_cast<const uint16_t *>(p + h.off_freq);
  uint32_t sum = 0;
  for (int s = 0; s < 256; ++s) {
    if (fq[s] >= kM) return ANSLIN_ERR_CORRUPT;
    sum += fq[s];
  }
  if (sum != kM) return ANSLIN_ERR_CORRUPT;
  const uint32_t *offs = reinterpret_cast<const uint32_t *>(p + h.off_offsets);
  uint64_t rec_end = is_bf16_like(g.fmt) ? h.off_raw : (h.off_scales ? h.off_scales : T);
  if (rec_end < h.off_records || rec_end > T) return ANSLIN_ERR_CORRUPT;
  const uint64_t rec_units = (rec_end - h.off_records) / 16;
  if (offs[0] != 0) return ANSLIN_ERR_CORRUPT;
  if (h.off_records + uint64_t(offs[g.n_tiles]) * 16 + kTailBytes > T) return ANSLIN_ERR_CORRUPT;  // tail rule
  for (size_t t = 0; t < g.n_tiles; ++t) {
    // a record holds at least the 32 lane states and never more than the worst-case tile
    if (offs[t + 1] < offs[t] + 8 || offs[t + 1] > rec_units) return ANSLIN_ERR_CORRUPT;
    if (uint64_t(offs[t + 1] - offs[t]) * 16 > 128 + uint64_t(g.steps) * kLanes * (g.fmt == ANSLIN_FMT_BF16_PAIR4 ? 6 : 2) + 16 + uint64_t(kSegTableBytes) * (g.steps / seg_steps_of(g.fmt) + 1))
      return ANSLIN_ERR_CORRUPT;
  }
  if (is_bf16_like(g.fmt) && !in(h.off_raw, raw_tile_bytes(g.tile_n, g.tile_k, g.flags) * g.n_tiles)) return ANSLIN_ERR_CORRUPT;
  if (g.fmt == ANSLIN_FMT_BF16_PAIR4 && !in(h.off_zeros, 16)) return ANSLIN_ERR_CORRUPT;
  if (side_bytes(g) && !in(h.off_scales, side_bytes(g))) return ANSLIN_ERR_CORRUPT;
  if ((g.flags & ANSLIN_FLAG_LANE_STREAMS) && (h.max_seg_bytes < 32 || h.max_seg_bytes > 2 * 0xFFFF + 64)) return ANSLIN_ERR_CORRUPT;
  // Lane-stream records: when the host copy includes the records section, every segment table is checked too (the kernels
  // turn its region sizes into shared-memory cursors): the region sizes add up to the segment's word count, the staged
  // segment fits the buffer the header promises (max_seg_bytes), and the segments stay inside their record.
  if ((g.flags & ANSLIN_FLAG_LANE_STREAMS) && bytes >= h.off_records + uint64_t(offs[g.n_tiles]) * 16) {
    const size_t nseg = size_t(g.steps) / seg_steps_of(g.fmt);
    for (size_t t = 0; t < g.n_tiles; ++t) {
      const uint8_t *rec = p + h.off_records + uint64_t(offs[t]) * 16;
      const uint64_t rec_bytes = uint64_t(offs[t + 1] - offs[t]) * 16;
      uint64_t goff = 4 * kLanes + uint64_t(kSegTableBytes) * nseg;
      if (goff > rec_bytes) return ANSLIN_ERR_CORRUPT;
      for (size_t sg = 0; sg < nseg; ++sg) {
        const uint8_t *te = rec + 4 * kLanes + kSegTableBytes * sg;
        uint16_t base, total;
        std::memcpy(&base, te, 2);
        std::memcpy(&total, te + 2, 2);
        uint32_t sum = 0;
        for (int r = 0; r < kLanes / 2; ++r) sum += uint32_t(base) + te[4 + r];
        if (sum != total) return ANSLIN_ERR_CORRUPT;
        const uint64_t staged = (((goff & 15) + 2 * uint64_t(total) + 15) & ~uint64_t(15));
        if (staged > align16(h.max_seg_bytes) || goff + 2 * uint64_t(total) > rec_bytes) return ANSLIN_ERR_CORRUPT;
        goff += 2 * uint64_t(total);
      }
    }
  }
  anslin_weight *w = new (std::nothrow) anslin_weight;
  if (!w) return ANSLIN_ERR_INVALID_ARG;
  w->h = h;
  w->dev = static_cast<const uint8_t *>(container_dev);
  *out = w;
  return ANSLIN_OK;
}

int anslin_close(anslin_weight *w) {
  delete w;
  return ANSLIN_OK;
}

int anslin_describe(const anslin_weight *w, anslin_desc *out) {
  if (!w || !out) return ANSLIN_ERR_INVALID_ARG;
  *out = anslin_desc{w->h.format, w->h.n_out, w->h.k_in, w->h.tile_k, w->h.group_size, w->h.flags, w->h.w_scale, w->h.tile_n};
  return ANSLIN_OK;
}

double anslin_entropy_bits(const uint64_t *counts_host, int32_t bins) {
  if (!counts_host || bins < 1) return 0.0;
  long double n = 0;
  for (int32_t i = 0; i < bins; ++i) n += counts_host[i];
  if (n == 0) return 0.0;
  long double h = 0;
  for (int32_t i = 0; i < bins; ++i)
    if (counts_host[i]) {
      const long double p = counts_host[i] / n;
      h -= p * log2l(p);
    }
  return double(h);
}

double anslin_entropy_weighted(const double *h, const uint64_t *n, int32_t layers) {
  if (!h || !n || layers < 1) return 0.0;
  long double num = 0, den = 0;
  for (int32_t i = 0; i < layers; ++i) { num += (long double)(n[i]) * h[i]; den += n[i]; }
  return den == 0 ? 0.0 : double(num / den);
}

const char *anslin_status_string(int s) {
  switch (s) {
    case ANSLIN_OK: return "ok";
    case ANSLIN_ERR_INVALID_ARG: return "invalid argument";
    case ANSLIN_ERR_UNSUPPORTED: return "unsupported shape or format";
    case ANSLIN_ERR_BUFFER_TOO_SMALL: return "buffer too small";
    case ANSLIN_ERR_CORRUPT: return "corrupt container";
    case ANSLIN_ERR_CUDA: return "CUDA error";
    case ANSLIN_ERR_STATIC_LIMIT: return "problem needs more scratch than the static workspace (ANSLIN_STATIC_WORKSPACE_BYTES) holds";
    default: return "unknown status";
  }
}

}  // extern "C"
