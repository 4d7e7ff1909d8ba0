// uts_scan.cuh — exclusive prefix sum of u32 counts into u64 offsets (used by the tile query and the radix sort).
// counts[n] -> offsets[n+1].  Three small kernels: per-block sums, scan of the block sums, per-block scan.  No spinning,
// no inter-block dependence inside a kernel.
#pragma once
#include "uts_internal.cuh"

namespace uts {

constexpr int kScanBlock = 256, kScanItems = 8, kScanTile = kScanBlock * kScanItems;

static __device__ __forceinline__ uint64_t block_exclusive_scan(uint64_t x, uint64_t* total_out) {
  __shared__ uint64_t wsum[kScanBlock / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint64_t incl = x;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { uint64_t y = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += y; }
  if (lane == 31) wsum[wid] = incl;
  __syncthreads();
  uint64_t before = 0, total = 0;
#pragma unroll
  for (int w = 0; w < kScanBlock / 32; ++w) { const uint64_t s = wsum[w]; if (w < wid) before += s; total += s; }
  __syncthreads();
  *total_out = total;
  return before + incl - x;
}

static __global__ void __launch_bounds__(kScanBlock) scan_block_sums(const uint32_t* __restrict__ counts, int64_t n, uint64_t* __restrict__ block_sums) {
  const int64_t base = (int64_t)blockIdx.x * kScanTile;
  uint64_t s = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) { const int64_t idx = base + j * kScanBlock + threadIdx.x; if (idx < n) s += counts[idx]; }
  uint64_t total;
  block_exclusive_scan(s, &total);
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

static __global__ void __launch_bounds__(kScanBlock) scan_of_sums(uint64_t* __restrict__ block_sums, int nb) {
  __shared__ uint64_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int b0 = 0; b0 < nb; b0 += kScanBlock) {
    const int b = b0 + threadIdx.x;
    const uint64_t x = b < nb ? block_sums[b] : 0;
    uint64_t total;
    const uint64_t ex = block_exclusive_scan(x, &total);
    if (b < nb) block_sums[b] = carry + ex;
    __syncthreads();
    if (threadIdx.x == 0) carry += total;
    __syncthreads();
  }
}

static __global__ void __launch_bounds__(kScanBlock) scan_write(const uint32_t* __restrict__ counts, int64_t n, const uint64_t* __restrict__ block_sums,
                                                         uint64_t* __restrict__ offsets) {
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;   // blocked arrangement
  uint32_t c[kScanItems];
  uint64_t s = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) { c[j] = (base + j < n) ? counts[base + j] : 0u; s += c[j]; }
  uint64_t total;
  uint64_t run = block_sums[blockIdx.x] + block_exclusive_scan(s, &total);
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) { if (base + j < n) offsets[base + j] = run; run += c[j]; }
  if (blockIdx.x == gridDim.x - 1) {
    __syncthreads();
    if (threadIdx.x == kScanBlock - 1) offsets[n] = block_sums[blockIdx.x] + total;
  }
}


inline size_t scan_scratch_bytes(int64_t n) { return (size_t)(((n + kScanTile - 1) / kScanTile + 1) * 8 + 256); }

// block_sums: scan_scratch_bytes(n) bytes of device scratch.
inline int exclusive_scan_u32(const uint32_t* counts, int64_t n, uint64_t* offsets, uint64_t* block_sums, cudaStream_t s) {
  if (n <= 0) { UTS_CUDA(cudaMemsetAsync(offsets, 0, sizeof(uint64_t), s)); return UTS_OK; }
  const int nb = (int)((n + kScanTile - 1) / kScanTile);
  scan_block_sums<<<nb, kScanBlock, 0, s>>>(counts, n, block_sums);
  UTS_LAUNCH_CHECK();
  scan_of_sums<<<1, kScanBlock, 0, s>>>(block_sums, nb);
  UTS_LAUNCH_CHECK();
  scan_write<<<nb, kScanBlock, 0, s>>>(counts, n, block_sums, offsets);
  UTS_LAUNCH_CHECK();
  return UTS_OK;
}

}  // namespace uts
