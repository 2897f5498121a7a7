// Internal definitions shared by the product's host encoder and device kernels (NOT by oracle/).
// Container byte layout: DESIGN.md §"Container".
#pragma once
#include <stdint.h>
#include <stddef.h>
#include "../../include/anslin.h"

#ifdef __CUDACC__
#define ANSLIN_HD __host__ __device__
#else
#define ANSLIN_HD
#endif

namespace anslin {

constexpr uint32_t kMagic = 0x4C534E41u;  // "ANSL"
constexpr uint32_t kVersion = 1;
constexpr int kTileN = 128;      // weight rows per stripe = tcgen05 MMA M; a stripe is cut into tiles of tile_n = 128 or 32 rows
constexpr int kLanes = 32;       // interleaved rANS streams per tile (P:l.192)
constexpr int kProbBits = 12;    // b (P:l.442)
constexpr int kWordBits = 16;    // w
constexpr int kStateLoLog2 = 16; // L = 2^16
constexpr uint32_t kL = 1u << kStateLoLog2;
constexpr uint32_t kM = 1u << kProbBits;
constexpr int kHeaderBytes = 128;
constexpr int kTailBytes = 4096; // readable bytes guaranteed after the records section (ring read-ahead)
constexpr int kSegTableBytes = 20; // per segment: u16 base, u16 total words, 16 x u8 (region words - base)
constexpr int kUnitBytes = 4096; // one operand unit = 128 rows x 32 B (one tcgen05.mma K step)

struct Header {  // 128 bytes, little endian
  uint32_t magic, version, format, n_out, k_in, tile_n, tile_k, streams, prob_bits, word_bits,
      state_lo_log2, group_size, flags, n_tiles;
  float w_scale;
  uint32_t max_seg_bytes;  // lane-stream layout: shared-memory bytes the largest segment needs when staged (else 0)
  uint64_t off_freq, off_offsets, off_records, off_raw, off_scales, off_zeros, total_bytes, reserved1;
};
static_assert(sizeof(Header) == kHeaderBytes, "header must be 128 bytes");

// symbols per 16-byte operand chunk
constexpr uint32_t kFormatMax = ANSLIN_FMT_BF16_PAIR4;
// stored as 16-bit bf16 values; the sign + mantissa byte of every weight lives in the raw plane
ANSLIN_HD constexpr bool is_bf16_like(uint32_t fmt) { return fmt == ANSLIN_FMT_BF16 || fmt == ANSLIN_FMT_BF16_PAIR4; }
// Decode steps per lane-stream segment (a segment is staged whole in shared memory, and costs a 20-byte table): 256 for the
// formats whose symbols carry few bits (bf16 exponents 2.6 bit, SQ8 4.5 bit), 128 where a symbol carries 6-7 bits (fp8, the
// packed 4-bit pairs, the bf16 exponent pairs) so that a staged segment stays near 3 KB and 16 decoder warps fit.
ANSLIN_HD constexpr int seg_steps_of(uint32_t fmt) { return (fmt == ANSLIN_FMT_BF16 || fmt == ANSLIN_FMT_INT8) ? 256 : 128; }
ANSLIN_HD constexpr bool is_fp8(uint32_t fmt) { return fmt == ANSLIN_FMT_FP8_E4M3 || fmt == ANSLIN_FMT_FP8_E5M2; }
// formats whose MMA runs in kind::f8f6f4 with a per-tensor weight scale and fp8 activations (fp4 is expanded to e4m3)
ANSLIN_HD constexpr bool is_fp8_path(uint32_t fmt) { return is_fp8(fmt) || fmt == ANSLIN_FMT_FP4_E2M1; }
// two 4-bit codes per coded byte
ANSLIN_HD constexpr bool is_packed4(uint32_t fmt) { return fmt == ANSLIN_FMT_INT4_AWQ || fmt == ANSLIN_FMT_FP4_E2M1; }
ANSLIN_HD constexpr int spc_of(uint32_t fmt) {
  return (fmt == ANSLIN_FMT_BF16 || fmt == ANSLIN_FMT_FP4_E2M1) ? 8 : (fmt == ANSLIN_FMT_INT4_AWQ || fmt == ANSLIN_FMT_BF16_PAIR4) ? 4 : 16;
}
ANSLIN_HD constexpr int weights_per_symbol(uint32_t fmt) { return (is_packed4(fmt) || fmt == ANSLIN_FMT_BF16_PAIR4) ? 2 : 1; }
// weights along K covered by one operand unit (32 bytes of bf16/fp16 = 16, of fp8/int8 = 32)
ANSLIN_HD constexpr int unit_k_of(uint32_t fmt) {
  return (is_bf16_like(fmt) || fmt == ANSLIN_FMT_INT4_AWQ) ? 16 : 32;
}
constexpr uint32_t default_tile_k(uint32_t fmt) { return fmt == ANSLIN_FMT_BF16 ? 64 : 256; }
// bytes per stored weight element of row-major W (int4: half a byte -> handled by callers)
ANSLIN_HD constexpr size_t raw_tile_bytes(uint32_t tile_n, uint32_t tile_k, uint32_t flags) {
  return size_t(tile_n) * tile_k - ((flags & ANSLIN_FLAG_STATE_PAYLOAD) ? 64 : 0);
}
inline size_t align16(size_t x) { return (x + 15) & ~size_t(15); }

}  // namespace anslin

struct anslin_weight {
  anslin::Header h;
  const uint8_t *dev;  // device copy of the whole container (may be null)
};
