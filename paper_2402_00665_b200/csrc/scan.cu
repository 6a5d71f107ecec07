// scan.cu -- K7: exclusive prefix sum of the per-query hit counts (int32) into 64-bit CSR offsets
// (count-then-fill; reading G21).  Reduce-then-scan: tile sums, a single-block scan of the tile sums,
// then each tile rescans itself from its base.  offsets[q] = nnz.
#include "common.cuh"

namespace bvh {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;

__device__ __forceinline__ int64_t block_exclusive_scan(int64_t v, int64_t* total, int64_t* s_warp) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int64_t incl = v;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const int64_t a = __shfl_up_sync(0xffffffffu, incl, off);
    if (lane >= off) incl += a;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  int64_t base = 0, sum = 0;
#pragma unroll
  for (int w = 0; w < kScanThreads / 32; ++w) {
    const int64_t s = s_warp[w];
    if (w < warp) base += s;
    sum += s;
  }
  __syncthreads();
  *total = sum;
  return base + incl - v;
}

__global__ void __launch_bounds__(kScanThreads) scan_tile_sums_kernel(const int32_t* __restrict__ counts, int64_t q,
                                                                      int64_t* __restrict__ tile_sums) {
  __shared__ int64_t s_warp[kScanThreads / 32];
  pdl_wait();
  pdl_trigger();
  const int64_t base = (int64_t)blockIdx.x * kScanTile;
  int64_t v = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    const int64_t i = base + k * kScanThreads + threadIdx.x;
    if (i < q) v += counts[i];
  }
  int64_t total;
  block_exclusive_scan(v, &total, s_warp);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanThreads) scan_of_sums_kernel(int64_t* tile_sums, int64_t tiles) {
  __shared__ int64_t s_warp[kScanThreads / 32];
  pdl_wait();
  pdl_trigger();
  int64_t carry = 0;
  for (int64_t b = 0; b < tiles; b += kScanThreads) {
    const int64_t i = b + threadIdx.x;
    const int64_t v = (i < tiles) ? tile_sums[i] : 0;
    int64_t total;
    const int64_t e = block_exclusive_scan(v, &total, s_warp);
    if (i < tiles) tile_sums[i] = carry + e;
    carry += total;
  }
}

__global__ void __launch_bounds__(kScanThreads) scan_apply_kernel(const int32_t* __restrict__ counts, int64_t q,
                                                                  const int64_t* __restrict__ tile_sums,
                                                                  int64_t* __restrict__ offsets) {
  __shared__ int64_t s_warp[kScanThreads / 32];
  pdl_wait();
  pdl_trigger();
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;  // blocked arrangement
  int32_t c[kScanItems];
  int64_t v = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    c[k] = (base + k < q) ? counts[base + k] : 0;
    v += c[k];
  }
  int64_t total;
  int64_t run = tile_sums[blockIdx.x] + block_exclusive_scan(v, &total, s_warp);
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    if (base + k < q) offsets[base + k] = run;
    run += c[k];
    if (base + k == q - 1) offsets[q] = run;
  }
}

// q <= kScanTile: the whole scan in one block (small batches are bound by the number of dependent launches).
__global__ void __launch_bounds__(kScanThreads) scan_single_tile_kernel(const int32_t* __restrict__ counts, int64_t q,
                                                                        int64_t* __restrict__ offsets) {
  __shared__ int64_t s_warp[kScanThreads / 32];
  pdl_wait();
  pdl_trigger();
  const int64_t base = (int64_t)threadIdx.x * kScanItems;   // blocked arrangement
  int32_t c[kScanItems];
  int64_t v = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    c[k] = (base + k < q) ? counts[base + k] : 0;
    v += c[k];
  }
  int64_t total;
  int64_t run = block_exclusive_scan(v, &total, s_warp);
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    if (base + k < q) offsets[base + k] = run;
    run += c[k];
  }
  if (threadIdx.x == 0) offsets[q] = total;
}

__global__ void scan_empty_kernel(int64_t* offsets) {
  pdl_wait();
  offsets[0] = 0;
}

size_t scan_scratch_bytes(int64_t q) {
  const int64_t tiles = (q + kScanTile - 1) / kScanTile;
  return (size_t)(tiles > 0 ? tiles : 1) * sizeof(int64_t);
}

cudaError_t launch_scan(const int32_t* counts, int64_t q, int64_t* offsets, void* scratch, cudaStream_t stream) {
  if (q == 0) return launch_pdl(scan_empty_kernel, dim3(1), dim3(1), 0, stream, offsets);
  if (q <= kScanTile) return launch_pdl(scan_single_tile_kernel, dim3(1), dim3(kScanThreads), 0, stream, counts, q, offsets);
  const int64_t tiles = (q + kScanTile - 1) / kScanTile;
  int64_t* sums = static_cast<int64_t*>(scratch);
  cudaError_t e = launch_pdl(scan_tile_sums_kernel, dim3((unsigned)tiles), dim3(kScanThreads), 0, stream, counts, q, sums);
  if (e == cudaSuccess) e = launch_pdl(scan_of_sums_kernel, dim3(1), dim3(kScanThreads), 0, stream, sums, tiles);
  if (e == cudaSuccess)
    e = launch_pdl(scan_apply_kernel, dim3((unsigned)tiles), dim3(kScanThreads), 0, stream, counts, q,
                   static_cast<const int64_t*>(sums), offsets);
  return e;
}

}  // namespace bvh
