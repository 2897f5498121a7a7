// Entropy-study histograms on the device (S: §8(f) NEXT-4; P:l.64-78 "we build an empirical histogram over these
// symbols and estimate the Shannon entropy", Fig. 2): 256-bin counts of the 8-bit symbols the coder sees (a1), taken
// from a row-major weight tensor resident in HBM.  HBM-bound by design: one pass, 16-byte loads, counters private to
// a (bin, lane) pair in shared memory so that the 32 lanes of a warp never collide on a bank.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/anslin.h"
#include "anslin_internal.h"

namespace anslin {
namespace {

constexpr int kHistThreads = 256;
constexpr int kPlaneWords = 256 * 32;   // [bin][lane] u32

__device__ __forceinline__ uint4 ldg128_nc(const uint4 *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}

// MODE 0: bf16 (plane 0 = exponent byte, plane 1 = mantissa<<1 | sign); 1: bytes (plane 0); 2: packed 4-bit codes
// (plane 0 = packed byte, plane 1 bins 0..15 = the 4-bit codes).
template <int MODE>
__device__ __forceinline__ void count_word(uint32_t *h, uint32_t lane, uint32_t v) {
  if constexpr (MODE == 0) {
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const uint32_t x = (v >> (16 * i)) & 0xFFFFu;
      atomicAdd(h + ((x >> 7) & 0xFFu) * 32 + lane, 1u);
      atomicAdd(h + kPlaneWords + ((((x & 0x7Fu) << 1) | (x >> 15)) * 32 + lane), 1u);
    }
  } else {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const uint32_t b = (v >> (8 * i)) & 0xFFu;
      atomicAdd(h + b * 32 + lane, 1u);
      if constexpr (MODE == 2) {
        atomicAdd(h + kPlaneWords + (b & 0xFu) * 32 + lane, 1u);
        atomicAdd(h + kPlaneWords + (b >> 4) * 32 + lane, 1u);
      }
    }
  }
}

template <int MODE>
__global__ void __launch_bounds__(kHistThreads) histogram_kernel(const uint4 *__restrict__ w, uint64_t n_vec, const uint8_t *__restrict__ tail,
                                                                 uint32_t n_tail, unsigned long long *__restrict__ counts) {
  extern __shared__ uint32_t h[];
  constexpr int kPlanes = MODE == 1 ? 1 : 2;
  for (int i = threadIdx.x; i < kPlanes * kPlaneWords; i += kHistThreads) h[i] = 0;
  __syncthreads();
  const uint32_t lane = threadIdx.x & 31;
  const uint64_t stride = uint64_t(gridDim.x) * kHistThreads;
  uint64_t i = uint64_t(blockIdx.x) * kHistThreads + threadIdx.x;
  for (; i + stride < n_vec; i += 2 * stride) {   // two loads in flight per thread
    const uint4 a = ldg128_nc(w + i), b = ldg128_nc(w + i + stride);
    count_word<MODE>(h, lane, a.x); count_word<MODE>(h, lane, a.y); count_word<MODE>(h, lane, a.z); count_word<MODE>(h, lane, a.w);
    count_word<MODE>(h, lane, b.x); count_word<MODE>(h, lane, b.y); count_word<MODE>(h, lane, b.z); count_word<MODE>(h, lane, b.w);
  }
  if (i < n_vec) {
    const uint4 a = ldg128_nc(w + i);
    count_word<MODE>(h, lane, a.x); count_word<MODE>(h, lane, a.y); count_word<MODE>(h, lane, a.z); count_word<MODE>(h, lane, a.w);
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {   // < 16 trailing bytes
    constexpr uint32_t kStep = MODE == 0 ? 2 : 1;
    for (uint32_t t = 0; t + kStep <= n_tail; t += kStep) {
      if constexpr (MODE == 0) {
        const uint32_t x = uint32_t(tail[t]) | (uint32_t(tail[t + 1]) << 8);
        atomicAdd(h + ((x >> 7) & 0xFFu) * 32, 1u);
        atomicAdd(h + kPlaneWords + (((x & 0x7Fu) << 1) | (x >> 15)) * 32, 1u);
      } else {
        const uint32_t b = tail[t];
        atomicAdd(h + b * 32, 1u);
        if constexpr (MODE == 2) {
          atomicAdd(h + kPlaneWords + (b & 0xFu) * 32, 1u);
          atomicAdd(h + kPlaneWords + (b >> 4) * 32, 1u);
        }
      }
    }
  }
  __syncthreads();
  // thread t sums bin t over the 32 lane columns (rotated start: no bank conflict) and adds it to the global count
  for (int p = 0; p < kPlanes; ++p) {
    const uint32_t *row = h + p * kPlaneWords + threadIdx.x * 32;
    unsigned long long s = 0;
#pragma unroll 8
    for (uint32_t k = 0; k < 32; ++k) s += row[(k + lane) & 31u];
    if (s) atomicAdd(counts + p * 256 + threadIdx.x, s);
  }
}

template <int MODE>
int launch_histogram(const void *w_dev, uint64_t n_bytes, unsigned long long *counts, cudaStream_t st) {
  static int sms = 0;
  if (sms == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
      sms = 0;
      return ANSLIN_ERR_CUDA;
    }
  }
  constexpr size_t smem = (MODE == 1 ? 1 : 2) * kPlaneWords * 4;
  auto kern = histogram_kernel<MODE>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess) return ANSLIN_ERR_CUDA;
  const int per_sm = MODE == 1 ? 6 : 3;
  // a (bin, lane) counter of one CTA is 32 bits: keep every launch below 2^31 symbols per CTA
  const uint64_t max_bytes = (uint64_t(1) << 30) * uint64_t(sms);
  const uint8_t *p = static_cast<const uint8_t *>(w_dev);
  for (uint64_t off = 0; off < n_bytes || off == 0; off += max_bytes) {
    const uint64_t nb = n_bytes - off < max_bytes ? n_bytes - off : max_bytes;
    const uint64_t n_vec = nb / 16;
    const uint64_t want = (n_vec + kHistThreads - 1) / kHistThreads;
    const uint32_t grid = uint32_t(want < uint64_t(sms * per_sm) ? (want ? want : 1) : uint64_t(sms * per_sm));
    kern<<<grid, kHistThreads, smem, st>>>(reinterpret_cast<const uint4 *>(p + off), n_vec, p + off + n_vec * 16, uint32_t(nb - n_vec * 16), counts);
    if (n_bytes == 0) break;
  }
  return cudaGetLastError() == cudaSuccess ? ANSLIN_OK : ANSLIN_ERR_CUDA;
}

}  // namespace
}  // namespace anslin

extern "C" int anslin_histogram(uint32_t format, const void *w_dev, uint64_t n_elems, void *counts_dev, void *stream) {
  using namespace anslin;
  if (!w_dev || !counts_dev || (reinterpret_cast<uintptr_t>(w_dev) & 15) || (reinterpret_cast<uintptr_t>(counts_dev) & 7)) return ANSLIN_ERR_INVALID_ARG;
  if (format > kFormatMax) return ANSLIN_ERR_UNSUPPORTED;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (cudaMemsetAsync(counts_dev, 0, 2 * 256 * sizeof(unsigned long long), st) != cudaSuccess) return ANSLIN_ERR_CUDA;
  unsigned long long *counts = static_cast<unsigned long long *>(counts_dev);
  if (format == ANSLIN_FMT_BF16) return launch_histogram<0>(w_dev, n_elems * 2, counts, st);
  if (is_packed4(format)) return launch_histogram<2>(w_dev, n_elems, counts, st);
  return launch_histogram<1>(w_dev, n_elems, counts, st);
}
