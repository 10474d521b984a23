// tpc_links.cuh -- a3 cleaner + start-hit finder   (O3; R8).  The neighbour finder is tpc_neighbours.cuh.
//
// All link arrays inside the library hold SORTED positions (the grid's order); the original input index
// (sorted_to_orig) enters only where the method defines a result through it: tie-breaks (R6) and the order
// of the start-hit list (R8).
#pragma once
#include "tpc_common.cuh"
#include "tpc_neighbours.cuh"

namespace tpc {

// thread per cluster.  O3: up'[h] = up[h] if dn[up[h]] == h else -1 (and symmetric); start hit <=> no down link
// and an up link.  The start flag is scattered to the ORIGINAL index so that the list comes out in ascending
// global input index (R8): spos_by_orig[orig] = sorted position, or -1 (array pre-set to -1).
__global__ void __launch_bounds__(256) cleanLinks(int64_t N, const int32_t* __restrict__ lup,
                                                  const int32_t* __restrict__ ldn, const uint32_t* __restrict__ s2o,
                                                  int32_t* __restrict__ cup, int32_t* __restrict__ cdn,
                                                  int32_t* __restrict__ spos_by_orig, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= N) return;
  const int32_t u = lup[p], d = ldn[p];
  const int32_t cu = (u >= 0 && __ldg(ldn + u) == (int32_t)p) ? u : -1;
  const int32_t cd = (d >= 0 && __ldg(lup + d) == (int32_t)p) ? d : -1;
  cup[p] = cu;
  cdn[p] = cd;
  if (cd == -1 && cu != -1) spos_by_orig[s2o[p]] = (int32_t)p;
}

// Stream compaction of the start hits in ascending original index, phase 1: per-tile counts.
constexpr int CP_THREADS = 256;
constexpr int CP_ITEMS = 8;
constexpr int CP_TILE = CP_THREADS * CP_ITEMS;

__global__ void __launch_bounds__(CP_THREADS) startCount(int64_t N, const int32_t* __restrict__ spos_by_orig,
                                                         uint32_t* __restrict__ tile_cnt) {
  __shared__ uint32_t sm[33];
  const int64_t first = (int64_t)blockIdx.x * CP_TILE + (int64_t)threadIdx.x * CP_ITEMS;
  uint32_t c = 0;
#pragma unroll
  for (int k = 0; k < CP_ITEMS; ++k)
    if (first + k < N && spos_by_orig[first + k] >= 0) ++c;
  uint32_t total;
  blockExclusiveScan(c, sm, &total);
  if (threadIdx.x == 0) tile_cnt[blockIdx.x] = total;
}

// phase 3 (after the tile offsets were scanned): write (orig index, sorted position) of every start hit.
__global__ void __launch_bounds__(CP_THREADS) startWrite(int64_t N, const int32_t* __restrict__ spos_by_orig,
                                                         const uint32_t* __restrict__ tile_off, int64_t cap,
                                                         uint32_t* __restrict__ start_orig,
                                                         uint32_t* __restrict__ start_pos) {
  __shared__ uint32_t sm[33];
  const int64_t first = (int64_t)blockIdx.x * CP_TILE + (int64_t)threadIdx.x * CP_ITEMS;
  int32_t v[CP_ITEMS];
  uint32_t c = 0;
#pragma unroll
  for (int k = 0; k < CP_ITEMS; ++k) {
    v[k] = (first + k < N) ? spos_by_orig[first + k] : -1;
    if (v[k] >= 0) ++c;
  }
  uint32_t total;
  uint32_t o = blockExclusiveScan(c, sm, &total) + tile_off[blockIdx.x];
#pragma unroll
  for (int k = 0; k < CP_ITEMS; ++k)
    if (v[k] >= 0) {
      if ((int64_t)o < cap) { start_orig[o] = (uint32_t)(first + k); start_pos[o] = (uint32_t)v[k]; }
      ++o;
    }
}

}  // namespace tpc
