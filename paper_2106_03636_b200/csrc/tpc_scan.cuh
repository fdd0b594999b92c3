// =============================================================================================
// tpc_scan.cuh -- device-wide exclusive prefix sum (int32 / int64), hand-written, three launches:
//   reduce   : one block per 4096-element tile -> tile sums
//   tiles    : one block scans the tile sums in place (exclusive), total appended
//   apply    : each block re-reads its tile, block-scans it, adds the tile offset, writes out
// Used for bin offsets (R7 `bin_first`), start-hit compaction (R10) and track/hit offsets (R20).
// No spin-waits and no inter-block dependencies inside a launch, so it cannot hang the device;
// the price is one extra read of the input (12 instead of 8 bytes per int32 element).
// =============================================================================================
#pragma once
#include "tpc_common.cuh"
#include "tpc_prof.cuh"

namespace tpc {

constexpr int kScanThreads = 256;
constexpr int kScanItems = kScanTile / kScanThreads;  // 16

template <class T>
__device__ __forceinline__ T warp_incl_scan(T v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    T o = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += o;
  }
  return v;
}

// exclusive scan of one value per thread across the block; returns exclusive prefix, *total = block sum
template <class T, int THREADS>
__device__ __forceinline__ T block_excl_scan(T v, T* total, T* smem /* THREADS/32 + 1 */) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const T inc = warp_incl_scan(v, lane);
  if (lane == 31) smem[w] = inc;
  __syncthreads();
  if (w == 0) {
    T s = (lane < THREADS / 32) ? smem[lane] : (T)0;
    const T si = warp_incl_scan(s, lane);
    if (lane < THREADS / 32) smem[lane] = si - s;
    if (lane == THREADS / 32 - 1) smem[THREADS / 32] = si;
  }
  __syncthreads();
  const T r = (inc - v) + smem[w];
  *total = smem[THREADS / 32];
  __syncthreads();
  return r;
}

template <class T>
__global__ void __launch_bounds__(kScanThreads) k_scan_reduce(const T* __restrict__ in, int64_t n, T* __restrict__ tile_sums) {
  __shared__ T sm[kScanThreads / 32 + 1];
  const int64_t base = (int64_t)blockIdx.x * kScanTile;
  T acc = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; k++) {
    const int64_t i = base + (int64_t)k * kScanThreads + threadIdx.x;
    if (i < n) acc += in[i];
  }
  T total;
  block_excl_scan<T, kScanThreads>(acc, &total, sm);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

template <class T>
__global__ void __launch_bounds__(1024) k_scan_tiles(T* __restrict__ tile_sums, int64_t ntiles) {
  __shared__ T sm[1024 / 32 + 1];
  T carry = 0;
  for (int64_t base = 0; base < ntiles; base += 1024) {
    const int64_t i = base + threadIdx.x;
    const T v = (i < ntiles) ? tile_sums[i] : (T)0;
    T total;
    const T ex = block_excl_scan<T, 1024>(v, &total, sm);
    if (i < ntiles) tile_sums[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0) tile_sums[ntiles] = carry;
}

// out may alias in.  Each thread owns kScanItems CONSECUTIVE elements so the scan order is the array order.
template <class T>
__global__ void __launch_bounds__(kScanThreads) k_scan_apply(const T* in, T* out, int64_t n, const T* __restrict__ tile_sums) {
  __shared__ T sm[kScanThreads / 32 + 1];
  __shared__ T tile[kScanTile + kScanTile / 16];  // +1 per 16: conflict-free for both access patterns
#define TPC_TI(j) ((j) + ((j) >> 4))
  const int64_t base = (int64_t)blockIdx.x * kScanTile;
#pragma unroll
  for (int k = 0; k < kScanItems; k++) {
    const int j = k * kScanThreads + threadIdx.x;
    const int64_t i = base + j;
    tile[TPC_TI(j)] = (i < n) ? in[i] : (T)0;
  }
  __syncthreads();
  T v[kScanItems];
  T acc = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; k++) {
    v[k] = tile[TPC_TI(threadIdx.x * kScanItems + k)];
    acc += v[k];
  }
  T total;
  T ex = block_excl_scan<T, kScanThreads>(acc, &total, sm) + tile_sums[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kScanItems; k++) {
    tile[TPC_TI(threadIdx.x * kScanItems + k)] = ex;
    ex += v[k];
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < kScanItems; k++) {
    const int j = k * kScanThreads + threadIdx.x;
    const int64_t i = base + j;
    if (i < n) out[i] = tile[TPC_TI(j)];
  }
#undef TPC_TI
}

// Exclusive scan of in[0..n) into out[0..n) (out may alias in); tmp holds >= ceil(n/4096)+1 elements.
// After completion tmp[ceil(n/4096)] holds the grand total.
template <class T>
inline cudaError_t exclusive_scan(const T* in, T* out, int64_t n, T* tmp, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  const int64_t ntiles = (n + kScanTile - 1) / kScanTile;
  TPC_LAUNCH(KID_SCAN, st, (k_scan_reduce<T><<<(unsigned)ntiles, kScanThreads, 0, st>>>(in, n, tmp)));
  TPC_LAUNCH(KID_SCAN, st, (k_scan_tiles<T><<<1, 1024, 0, st>>>(tmp, ntiles)));
  TPC_LAUNCH(KID_SCAN, st, (k_scan_apply<T><<<(unsigned)ntiles, kScanThreads, 0, st>>>(in, out, n, tmp)));
  return cudaGetLastError();
}

}  // namespace tpc
