// tpc_scan.cuh -- block / device exclusive prefix sums used by the grid build and the compactions.
// Three phases (tile sums -> scan of the tile sums by one block -> apply); no inter-block waiting, so the
// kernels can never hang on scheduling order.  The element count lives on the device (a counter written by
// an earlier kernel of the same stream): blocks beyond it exit at once.
#pragma once
#include "tpc_common.cuh"

namespace tpc {

constexpr int SCAN_THREADS = 512;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

template <typename T>
__device__ __forceinline__ T warpInclusiveScan(T v) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    T o = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += o;
  }
  return v;
}

// exclusive scan of one value per thread over the block; returns the exclusive prefix, *total = block sum.
// smem: at least 33 elements of T.  Ends with a __syncthreads() so smem can be reused.
template <typename T>
__device__ __forceinline__ T blockExclusiveScan(T v, T* smem, T* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
  const T inc = warpInclusiveScan(v);
  if (lane == 31) smem[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    T w = lane < nwarp ? smem[lane] : T(0);
    T winc = warpInclusiveScan(w);
    smem[lane] = winc - w;
    if (lane == 31) smem[32] = winc;
  }
  __syncthreads();
  const T res = smem[warp] + inc - v;
  *total = smem[32];
  __syncthreads();
  return res;
}

template <typename T>
__global__ void __launch_bounds__(SCAN_THREADS) scanTileSums(const T* __restrict__ in, const int64_t* __restrict__ n_dev,
                                                             int64_t n_cap, T* __restrict__ tile_sum) {
  __shared__ T sm[33];
  const int64_t n = min(*n_dev, n_cap);
  const int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
  if (base >= n) return;
  T s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    const int64_t i = base + (int64_t)k * SCAN_THREADS + threadIdx.x;
    if (i < n) s += in[i];
  }
  T total;
  blockExclusiveScan(s, sm, &total);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

// one block: exclusive scan of the tile sums in place; grand total -> *total_out (if not NULL)
template <typename T>
__global__ void __launch_bounds__(1024) scanTileOffsets(T* __restrict__ tile_sum, const int64_t* __restrict__ n_dev,
                                                        int64_t n_cap, T* __restrict__ total_out) {
  __shared__ T sm[33];
  const int64_t n = min(*n_dev, n_cap);
  const int64_t ntiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  T carry = 0;
  for (int64_t base = 0; base < ntiles; base += blockDim.x) {
    const int64_t i = base + threadIdx.x;
    const T v = i < ntiles ? tile_sum[i] : T(0);
    T total;
    const T ex = blockExclusiveScan(v, sm, &total);
    if (i < ntiles) tile_sum[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0 && total_out) *total_out = carry;
}

// out[i] = exclusive prefix of in[0..i); out[n] = total (sentinel).  in == out is allowed.
template <typename T>
__global__ void __launch_bounds__(SCAN_THREADS) scanApply(const T* in, T* out, const int64_t* __restrict__ n_dev,
                                                          int64_t n_cap, const T* __restrict__ tile_off) {
  __shared__ T sm[33];
  const int64_t n = min(*n_dev, n_cap);
  const int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
  if (base >= n) {
    if (base == 0 && threadIdx.x == 0) out[0] = 0;   // n == 0: only the sentinel
    return;
  }
  // blocked arrangement: thread t owns items [t*ITEMS, (t+1)*ITEMS) of the tile
  T v[SCAN_ITEMS];
  T s = 0;
  const int64_t first = base + (int64_t)threadIdx.x * SCAN_ITEMS;
  // a thread's items are SCAN_ITEMS * sizeof(T) consecutive bytes: 16-byte loads and stores wherever the whole run is
  // inside the array and the arrays are 16-byte aligned (always, for the workspace arrays of this library)
  constexpr int VEC = 16 / sizeof(T);
  const bool whole = first + SCAN_ITEMS <= n && ((reinterpret_cast<uintptr_t>(in) | reinterpret_cast<uintptr_t>(out)) & 15) == 0;
  if (whole) {
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k += VEC) {
      const uint4 q = *reinterpret_cast<const uint4*>(in + first + k);
      memcpy(&v[k], &q, 16);
    }
  } else {
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) v[k] = (first + k < n) ? in[first + k] : T(0);
  }
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) s += v[k];
  T total;
  T ex = blockExclusiveScan(s, sm, &total) + tile_off[blockIdx.x];
  if (whole) {
    T o[SCAN_ITEMS];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { o[k] = ex; ex += v[k]; }
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k += VEC) {
      uint4 q;
      memcpy(&q, &o[k], 16);
      *reinterpret_cast<uint4*>(out + first + k) = q;
    }
    if (first + SCAN_ITEMS == n) out[n] = ex;
  } else {
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
      if (first + k < n) out[first + k] = ex;
      ex += v[k];
      if (first + k == n - 1) out[n] = ex;
    }
  }
}

}  // namespace tpc

namespace tpc {
// one block: exclusive scan of a[0..n) in place (n known on the host); total -> *total_out (int64 counter)
template <typename T>
__global__ void __launch_bounds__(1024) scanArrayInPlace(T* __restrict__ a, int64_t n, int64_t* __restrict__ total_out) {
  __shared__ T sm[33];
  T carry = 0;
  for (int64_t base = 0; base < n; base += blockDim.x) {
    const int64_t i = base + threadIdx.x;
    const T v = i < n ? a[i] : T(0);
    T total;
    const T ex = blockExclusiveScan(v, sm, &total);
    if (i < n) a[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0 && total_out) *total_out = (int64_t)carry;
}
}  // namespace tpc
