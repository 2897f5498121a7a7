/*
 * anslin.h — C ABI of libanslin: tile-level rANS weight compression fused into tcgen05 GEMM on B200.
 *
 * Follows the problem statement of arxiv/paper_2606_15789 (P = /root/reference/PAPER.md):
 *   offline: compress each projection matrix into tile-aligned, independently decodable rANS
 *            substreams with one shared per-matrix codebook and a 4-byte offset per tile
 *            (P:l.149 §IV-A, P:l.165-169 §V-B, Eq.3 P:l.440);
 *   run time: decode tiles on the SMs straight into shared memory and feed the tensor cores
 *            (P:l.181-252 Alg V.1, P:l.260-287 Alg V.2, P:l.301-304 Alg V.3), or decode only.
 *
 * Conventions (all entry points):
 *   - return value: anslin_status (0 = ANSLIN_OK); no exceptions, no abort, nothing printed.
 *   - "host" pointers are CPU memory, "dev" pointers are CUDA device memory of the current device.
 *   - the CALLER owns every buffer; the library allocates no device memory and keeps no global
 *     state.  Handles (anslin_weight) are small host objects released with anslin_close.
 *   - kernels are enqueued on the caller's stream and run asynchronously; asynchronous faults
 *     surface at the caller's next synchronisation.  No hidden synchronisation.
 *   - device pointers must be 16-byte aligned (else ANSLIN_ERR_INVALID_ARG).
 *   - shapes: n_out % 128 == 0 and k_in % tile_k == 0 (else ANSLIN_ERR_UNSUPPORTED); m >= 1 (anslin_gemm_multi: <= 256 per problem).
 *   - orientation: W is [n_out x k_in] row-major (torch Linear.weight), X is [m x k_in] row-major
 *     with leading dimension ldx (elements), Y is [m x n_out] row-major float32 with ldy.
 *   - there is no CPU fallback: the device entry points fail with ANSLIN_ERR_CUDA when no sm_100
 *     device / driver is usable.
 *
 * The byte layout of a container is specified in DESIGN.md §"Container".
 */
#ifndef ANSLIN_H
#define ANSLIN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  ANSLIN_OK = 0,
  ANSLIN_ERR_INVALID_ARG = 1,
  ANSLIN_ERR_UNSUPPORTED = 2,
  ANSLIN_ERR_BUFFER_TOO_SMALL = 3,
  ANSLIN_ERR_CORRUPT = 4,
  ANSLIN_ERR_CUDA = 5,
  ANSLIN_ERR_STATIC_LIMIT = 6   /* anslin_gemm_static: the problem needs more scratch than the library's static array holds */
} anslin_status;

/* Numeric format of W (P:l.80, l.341; BASELINE.json configs 1-5). */
typedef enum {
  ANSLIN_FMT_BF16 = 0,     /* w_host: uint16 bit patterns; coded symbol = exponent byte, sign+mantissa raw */
  ANSLIN_FMT_FP8_E4M3 = 1, /* w_host: e4m3fn bytes; coded symbol = the byte; per-tensor scale in desc.w_scale */
  ANSLIN_FMT_INT8 = 2,     /* w_host: int8; coded symbol = the byte; scales_host = fp16[n_out] (SQ8-style) */
  ANSLIN_FMT_INT4_AWQ = 3, /* w_host: uint8[n_out][k_in/2], low nibble = even k; coded symbol = packed byte;
                              scales_host/zeros_host = fp16[n_out][k_in/group_size]; w = (q - z) * s.
                              Plain per-channel int4 is this format with group_size = k_in (symmetric: z = 8) */
  ANSLIN_FMT_FP8_E5M2 = 4, /* w_host: OCP e5m2 bytes (P:l.80 "FP8-E5M2"); otherwise as FP8_E4M3 */
  ANSLIN_FMT_FP4_E2M1 = 5, /* w_host: uint8[n_out][k_in/2], low nibble = even k, OCP e2m1 codes s.ee.m (P:l.80 "FP4-E2M1");
                              coded symbol = packed byte; per-tensor scale in desc.w_scale.  Every code is expanded
                              exactly to e4m3 for the tensor core; X is fp8 (either kind) with per-token scales */
  ANSLIN_FMT_BF16_PAIR4 = 6 /* VARIANT of BF16 (S: NEXT-5), not the paper's symbolisation: the 15 most frequent exponent
                              bytes get 4-bit codes, code 15 = escape; coded symbol = the codes of two K-adjacent
                              weights, so one rANS step decodes two weights.  An escaped exponent follows as a literal
                              16-bit word in the lane's own stream.  Raw plane, payload flag, X and Y as BF16.
                              Lane-stream layout on 32-row tiles only (segments of 128 steps) */
} anslin_format;

/* Element type of X. */
typedef enum {
  ANSLIN_DT_F32 = 0, ANSLIN_DT_F16 = 1, ANSLIN_DT_BF16 = 2, ANSLIN_DT_I8 = 3, ANSLIN_DT_FP8_E4M3 = 4,
  ANSLIN_DT_FP8_E5M2 = 5
} anslin_dtype;

/* Container flag bits. */
#define ANSLIN_FLAG_STATE_PAYLOAD 1u /* bf16: each lane's rANS start state carries its last two raw-plane
                                        bytes ("arbitrary initial states", P:l.167; A4) */

#define ANSLIN_FLAG_LANE_STREAMS 2u  /* 32-row tiles only: every lane's 16-bit words are stored as a stream of its own
                                        (two lanes share a region, one ascending, one descending; 20 bytes of region
                                        sizes per segment = 256 decode steps for bf16 / int8, 128 for the other formats) instead of interleaved in read order: the decoder
                                        needs no ballot / prefix count.  Costs ~0.02 bit/weight.  If a tile cannot be
                                        represented (region sizes spread over > 255 words) the encoder silently drops
                                        the flag; anslin_describe reports the flags actually used. */

/* What the caller states about W. */
typedef struct {
  uint32_t format;      /* anslin_format */
  uint32_t n_out, k_in; /* W is [n_out x k_in] */
  uint32_t tile_k;      /* K extent of one tile in weights; 0 = format default (bf16 64, fp8/int8/int4 256);
                           32 interleaved streams per tile */
  uint32_t group_size;  /* int4: quantisation group along K (multiple of 16); else 0 */
  uint32_t flags;       /* ANSLIN_FLAG_* */
  float    w_scale;     /* fp8: per-tensor dequant scale applied to Y; other formats: ignored (1.0) */
  uint32_t tile_n;      /* weight rows per tile: 128 (= tcgen05 MMA M; 0 selects it; BASELINE config 1's 128 x 64)
                           or 32 (the paper's 32-row tile shape, P:l.444: four tiles share one MMA stripe) */
} anslin_desc;

/* Size accounting filled by the encoder (P:l.444 reports payload and metadata separately). Bits. */
typedef struct {
  uint64_t n_weights;
  uint64_t payload_bits;      /* rANS words */
  uint64_t state_bits;        /* 32 x 32-bit lane states per tile */
  uint64_t pad_bits;          /* 16-byte record padding */
  uint64_t offset_table_bits; /* 4 B per tile (+1 sentinel): Eq.3 first term */
  uint64_t freq_table_bits;   /* 256 x u16 */
  uint64_t raw_bits;          /* bf16 sign+mantissa plane */
  uint64_t side_bits;         /* scales / zeros (reported separately from bits/weight) */
  uint64_t total_bytes;
  double entropy_bits_per_symbol; /* H of the coded-symbol histogram (P:l.70) */
  double xent_bits_per_symbol;    /* cross entropy under the 12-bit table */
  double raw_entropy_bits_per_symbol; /* bf16 raw plane's own order-0 entropy, else 0 */
  double bits_per_weight;         /* 8 * (total_bytes - side bytes) / n_weights */
} anslin_stats;

/* Worst-case container size in bytes for `desc` (0 if desc is invalid). Host only. */
size_t anslin_encode_bound(const anslin_desc *desc);

/*
 * Offline CPU encoder and tile packer (P:l.165-169): histogram over the whole matrix, 12-bit
 * normalisation, per-tile 32-lane interleaved rANS with 16-bit words and 32-bit states.
 *   w_host, scales_host, zeros_host: host, read only (see anslin_format for shapes).
 *   container_out: host, capacity bytes; *bytes_out = bytes written.  stats_or_null: host.
 * Errors: INVALID_ARG (null/desc), UNSUPPORTED (shape/format), BUFFER_TOO_SMALL.
 */
int anslin_encode_host(const anslin_desc *desc, const void *w_host, const void *scales_host,
                       const void *zeros_host, void *container_out, size_t capacity,
                       size_t *bytes_out, anslin_stats *stats_or_null);

/* Host handle over a container whose bytes the caller has placed in device memory. */
typedef struct anslin_weight anslin_weight;

/*
 * Validate a container and bind it to its device copy.
 *   container_host: host copy (at least header + freq + offset sections; `bytes` = how many are
 *   readable); container_dev: device copy of the WHOLE container (16-byte aligned), may be NULL
 *   for host-only inspection.  Checks magic/version/shape/section bounds, that the frequency table
 *   sums to 2^12, that tile offsets are monotone and in range and -- when `bytes` covers the records
 *   section of a lane-stream container -- every segment table (region sizes add up to the segment's
 *   word count, the staged segment fits max_seg_bytes and its record) -> ANSLIN_ERR_CORRUPT otherwise.
 *   What anslin_open has checked cannot steer a kernel out of bounds.  A container whose records were
 *   never on the host (anslin_encode_device) is trusted; the kernels clamp every cursor they derive
 *   from a segment table into the staged buffer, so a damaged table there gives wrong weights.
 */
int anslin_open(const void *container_host, size_t bytes, const void *container_dev, anslin_weight **out);
int anslin_close(anslin_weight *w);
/* Copy of the descriptor the container was encoded with (tile_k resolved). */
int anslin_describe(const anslin_weight *w, anslin_desc *out);

/*
 * Decode only, to HBM (the paper's unfused stage, Fig. 9 P:l.410): writes W row-major in its
 * original dtype/packing to w_out_dev (capacity >= n_out*k_in*bytes_per_weight).
 * `stream` is a cudaStream_t passed as void*.
 */
int anslin_decode(const anslin_weight *w, void *w_out_dev, size_t capacity, void *stream);

/* Scratch bytes anslin_gemm needs for batch m (split-K partials + counters). */
size_t anslin_gemm_workspace_bytes(const anslin_weight *w, int32_t m);
/* Scratch bytes anslin_gemm_multi / anslin_gemm_grouped need for these n weights at batch sizes <= m_max. */
size_t anslin_gemm_multi_workspace_bytes(const anslin_weight *const *weights, int32_t n, int32_t m_max);

/*
 * Fused decode + GEMM, Y = X . W^T (Alg V.1): only compressed bytes of W cross HBM.
 *   x_dev: [m x k_in], dtype per format: bf16 -> BF16, int4 -> F16, int8 -> I8, fp8 (either kind) -> FP8_E4M3
 *   or FP8_E5M2 (the tensor core multiplies the two fp8 kinds in any combination).
 *   x_scale_dev: int8/fp8: f32[m] per-token scales; else NULL.
 *   y_dev: f32 [m x n_out]; int8: acc * x_scale[m] * w_scale[n]; fp8: acc * x_scale[m] * desc.w_scale.
 *   The launch may be captured in a CUDA graph and replayed (workspace and buffers must stay where they were).
 *   m >= 1.  m <= 256 is the regime the kernel is built for (P:l.295-306).  A larger m is processed in blocks of 256 rows,
 *   every block a problem of its own in one persistent launch (8 blocks per launch): each block decodes W again.
 */
int anslin_gemm(const anslin_weight *w, const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m,
                const void *x_scale_dev, void *y_dev, int64_t ldy, void *workspace_dev,
                size_t workspace_bytes, void *stream);

/*
 * anslin_gemm for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc)
 * and so cannot provide a workspace: the split-K scratch is a static device array inside the library
 * (ANSLIN_STATIC_WORKSPACE_BYTES, held by every GPU that loads the library until the process exits).  The call allocates
 * nothing: no cudaMalloc, cudaFree or allocating library routine; it enqueues one cudaMemsetAsync of the flag words and the
 * launch(es) of anslin_gemm on `stream`.  Arguments, layouts and results are anslin_gemm's.
 *   Limit: anslin_gemm_workspace_bytes(w, m) <= ANSLIN_STATIC_WORKSPACE_BYTES, else ANSLIN_ERR_STATIC_LIMIT and nothing is
 *   enqueued (24 MiB covers every shape at m <= 32 for containers the tensor-memory kernel takes; larger batches need
 *   anslin_gemm with a caller-owned workspace).
 *   The array is ONE per device and shared by every call: two calls that may overlap on the GPU (different streams, or
 *   graph branches without an edge between them) race on it and give wrong results; calls on one stream are ordered and safe.
 */
#define ANSLIN_STATIC_WORKSPACE_BYTES (24u << 20)
int anslin_gemm_static(const anslin_weight *w, const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m,
                       const void *x_scale_dev, void *y_dev, int64_t ldy, void *stream);

/*
 * n independent fused decode-GEMMs in ONE persistent launch (projections that share an input, e.g.
 * q/k/v or gate/up; the building block of anslin_gemm_grouped): Y_i = X_i . W_i^T.  The SMs are shared
 * out in proportion to n_out*k_in of each problem.  All weights must have the same format, tile_n and
 * state-payload flag; shapes, tile_k and batch sizes may differ.  Arrays are host arrays of n entries
 * (device pointers inside); x_scale_dev may be NULL for bf16 / int4.  More than 8 problems are issued
 * as consecutive launches on the same stream.  Workspace: anslin_gemm_multi_workspace_bytes.
 */
int anslin_gemm_multi(const anslin_weight *const *weights, int32_t n, const void *const *x_dev,
                      uint32_t x_dtype, const int64_t *ldx, const int32_t *m,
                      const void *const *x_scale_dev, void *const *y_dev, const int64_t *ldy,
                      void *workspace_dev, size_t workspace_bytes, void *stream);
/* The same with the element type of every Y chosen: ANSLIN_DT_F32 (as anslin_gemm_multi) or ANSLIN_DT_BF16 (the fp32
 * result rounded to nearest even; ldy in elements of that type; rows 8-byte aligned for vector stores, else scalar). */
int anslin_gemm_multi_ex(const anslin_weight *const *weights, int32_t n, const void *const *x_dev,
                         uint32_t x_dtype, const int64_t *ldx, const int32_t *m,
                         const void *const *x_scale_dev, void *const *y_dev, uint32_t y_dtype,
                         const int64_t *ldy, void *workspace_dev, size_t workspace_bytes, void *stream);

/*
 * Grouped fused decode-GEMM over MoE experts (BASELINE config 5): rows of X already sorted by
 * expert and contiguous; expert e owns rows_per_expert_host[e] rows (0 = inactive, skipped).
 * All experts share one shape/format.  Y rows are in the same order as X rows.  The active experts
 * run as the problems of one persistent launch (a12; table residency per CTA, one expert per CTA).
 * Workspace: anslin_gemm_multi_workspace_bytes(experts, n_experts, max rows of one expert).
 */
int anslin_gemm_grouped(const anslin_weight *const *experts, int32_t n_experts,
                        const int32_t *rows_per_expert_host, const void *x_dev, uint32_t x_dtype,
                        int64_t ldx, const void *x_scale_dev, void *y_dev, int64_t ldy,
                        void *workspace_dev, size_t workspace_bytes, void *stream);

/*
 * Uncompressed comparator: the same tcgen05 pipeline with TMA loads of raw W instead of decoder
 * warps ("uncompressed cuBLAS-free dense GEMM", BASELINE.json north_star).  w_dev: row-major W
 * in the operand dtype (bf16 / fp16 / int8 / e4m3; int4 is not supported here).
 */
size_t anslin_dense_workspace_bytes(uint32_t n_out, uint32_t k_in, int32_t m);
int anslin_dense_gemm(uint32_t format, const void *w_dev, uint32_t n_out, uint32_t k_in,
                      const void *w_scale_dev /* int8: fp16[n_out]; else NULL */, float w_scale,
                      const void *x_dev, uint32_t x_dtype, int64_t ldx, int32_t m,
                      const void *x_scale_dev, void *y_dev, int64_t ldy, void *workspace_dev,
                      size_t workspace_bytes, void *stream);

/*
 * Entropy study (P:l.64-78, Fig. 2; S: NEXT-4): empirical 256-bin histograms of the 8-bit symbols of a row-major
 * weight tensor resident in HBM, with the coder's own symbolisation (a1).
 *   w_dev: 16-byte aligned; n_elems = stored elements (bf16: 16-bit values; every other format: bytes).
 *   counts_dev: uint64[2][256], overwritten.  Plane 0 = coded symbols (bf16: exponent byte; fp8/int8: the byte;
 *   int4/fp4: the packed byte of two codes).  Plane 1 = bf16: the raw byte (mantissa<<1 | sign); int4/fp4: the 4-bit
 *   codes in bins 0..15; else zeros.  One pass over W, enqueued on `stream`; no synchronisation.
 */
int anslin_histogram(uint32_t format, const void *w_dev, uint64_t n_elems, void *counts_dev, void *stream);
/* H = -sum p log2 p of a histogram of `bins` host counts (P:l.70), bits per symbol; 0 for an empty histogram. */
double anslin_entropy_bits(const uint64_t *counts_host, int32_t bins);
/* Symbol-weighted model entropy (P:l.74): sum_l n[l] * h[l] / sum_l n[l]; 0 if all n are 0. */
double anslin_entropy_weighted(const double *h, const uint64_t *n, int32_t layers);

/*
 * GPU-side encoder (S: NEXT-6; the paper names it as future work, P:l.486): compress a row-major W that is resident
 * in HBM into a container in HBM.  Same symbolisation, table normalisation, container layout and decoders as
 * anslin_encode_host; restricted to the lane-stream layout (desc.tile_n = 32, ANSLIN_FLAG_LANE_STREAMS set, tile_k a
 * whole number of segments: a multiple of 256 weights for bf16 / int8 / int4 / fp4, of 128 for fp8).  An offline-stage call like
 * anslin_encode_host: it SYNCHRONISES `stream` (the 256-bin histogram and the per-tile record sizes visit the host
 * for the table normalisation and the offset prefix sum; W itself never leaves the device).
 *   w_dev: row-major W as anslin_encode_host takes it, 16-byte aligned.  scales_host / zeros_host: as anslin_encode_host.
 *   container_dev: >= anslin_encode_bound(desc) bytes.  head_host: >= anslin_encode_device_head_bytes(desc) bytes; receives
 *   the header, frequency table and record offsets — what anslin_open needs as `container_host`.
 *   workspace_dev: >= anslin_encode_device_workspace_bytes(desc) bytes.  *bytes_out = container size.
 * ANSLIN_ERR_UNSUPPORTED if the geometry is not the one above or a tile does not fit the lane-stream segment tables
 * (anslin_encode_host falls back to interleaved words in that case; this call does not).
 */
size_t anslin_encode_device_workspace_bytes(const anslin_desc *desc);
size_t anslin_encode_device_head_bytes(const anslin_desc *desc);
int anslin_encode_device(const anslin_desc *desc, const void *w_dev, const void *scales_host, const void *zeros_host,
                         void *container_dev, size_t capacity, void *head_host, size_t head_capacity,
                         void *workspace_dev, size_t workspace_bytes, size_t *bytes_out, void *stream);

/* How many kernels a GEMM call enqueues, as a function of its shape (the library keeps no state to ask): row_blocks = the
 * call's problems cut into blocks of at most 256 batch rows (anslin_gemm: ceil(m / 256); anslin_gemm_multi: n; grouped: sum
 * over active experts of ceil(rows / 256)); a launch takes up to eight blocks.  Host only. */
int anslin_gemm_launches(int64_t row_blocks);

const char *anslin_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* ANSLIN_H */
