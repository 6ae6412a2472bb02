// vd_scan.cuh -- device-wide exclusive prefix sum (used by S1 bucketing and S6 compaction).
// out[0..n] receives the exclusive scan of in[0..n-1]; out[n] = total.  Three launches:
// tile sums, scan of tile sums (one block), tile scans with carry-in.  HBM-bound streaming.
#pragma once
#include "vd_common.cuh"

namespace vd {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;

template <typename T>
__device__ __forceinline__ T block_exclusive_scan(T v, T* total) {
  // v: per-thread value; returns exclusive prefix within the block; *total = block sum
  __shared__ long long warpSum[kScanThreads / kLanes + 1];
  const int lane = lane_id(), w = (int)threadIdx.x / kLanes;
  T inc = v;
#pragma unroll
  for (int off = 1; off < kLanes; off <<= 1) {
    const T o = __shfl_up_sync(kFull, inc, off);
    if (lane >= off) inc += o;
  }
  if (lane == kLanes - 1) warpSum[w] = (long long)inc;
  __syncthreads();
  if (threadIdx.x == 0) {
    long long run = 0;
    const int nw = (int)blockDim.x / kLanes;
    for (int k = 0; k < nw; ++k) { const long long t = warpSum[k]; warpSum[k] = run; run += t; }
    warpSum[nw] = run;
  }
  __syncthreads();
  const T res = (T)warpSum[w] + inc - v;
  *total = (T)warpSum[(int)blockDim.x / kLanes];
  __syncthreads();
  return res;
}

template <typename TIn, typename TOut>
__global__ void __launch_bounds__(kScanThreads) scan_tile_sums(const TIn* __restrict__ in, int64_t n, TOut* __restrict__ tileSum) {
  const int64_t base = (int64_t)blockIdx.x * kScanTile;
  TOut s = 0;
  for (int k = 0; k < kScanItems; ++k) {
    const int64_t idx = base + (int64_t)k * kScanThreads + threadIdx.x;
    if (idx < n) s += (TOut)in[idx];
  }
  TOut total;
  block_exclusive_scan<TOut>(s, &total);
  if (threadIdx.x == 0) tileSum[blockIdx.x] = total;
}

template <typename TOut>
__global__ void __launch_bounds__(kScanThreads) scan_tile_offsets(TOut* __restrict__ tileSum, int64_t ntiles) {
  __shared__ long long carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int64_t base = 0; base < ntiles; base += kScanThreads) {
    const int64_t idx = base + threadIdx.x;
    const TOut v = idx < ntiles ? tileSum[idx] : (TOut)0;
    TOut total;
    const TOut ex = block_exclusive_scan<TOut>(v, &total);
    if (idx < ntiles) tileSum[idx] = ex + (TOut)carry;
    __syncthreads();
    if (threadIdx.x == 0) carry += (long long)total;
    __syncthreads();
  }
  if (threadIdx.x == 0) tileSum[ntiles] = (TOut)carry;
}

template <typename TIn, typename TOut>
__global__ void __launch_bounds__(kScanThreads) scan_tiles(const TIn* __restrict__ in, int64_t n, const TOut* __restrict__ tileSum,
                                                           TOut* __restrict__ out) {
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
  TOut v[kScanItems];
  TOut s = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    v[k] = (base + k < n) ? (TOut)in[base + k] : (TOut)0;
    s += v[k];
  }
  TOut total;
  TOut ex = block_exclusive_scan<TOut>(s, &total) + tileSum[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    if (base + k < n) out[base + k] = ex;
    ex += v[k];
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) out[n] = tileSum[gridDim.x];
}

// scratch must hold (ntiles + 1) TOut.  in and out may alias only if TIn == TOut (each thread
// reads its items before writing them).
template <typename TIn, typename TOut>
inline void exclusive_scan(const TIn* in, int64_t n, TOut* out, TOut* scratch, cudaStream_t stream) {
  const int64_t ntiles = (n + kScanTile - 1) / kScanTile;
  if (n <= 0) { cudaMemsetAsync(out, 0, sizeof(TOut), stream); return; }
  VD_LAUNCH((scan_tile_sums<TIn, TOut>), (unsigned)ntiles, kScanThreads, 0, stream)(in, n, scratch);
  VD_LAUNCH((scan_tile_offsets<TOut>), 1, kScanThreads, 0, stream)(scratch, ntiles);
  VD_LAUNCH((scan_tiles<TIn, TOut>), (unsigned)ntiles, kScanThreads, 0, stream)(in, n, scratch, out);
}

inline int64_t scan_scratch_elems(int64_t n) { return (n + kScanTile - 1) / kScanTile + 2; }

}  // namespace vd
