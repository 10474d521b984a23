// tpc_common.cuh -- device-side structs and small helpers shared by the kernels of libtpcgpu.so.
//
// Everything here is written from DESIGN.md section 3 (formula sheet).  No file under oracle/ is included.
// All selection / Kalman arithmetic is IEEE binary32, one rounding per written operation: this translation
// unit is compiled with --fmad=false -prec-div=true -prec-sqrt=true -ftz=false (R0).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tpc {

// Per (sector,row) bucket grid descriptor (O1).  Cells are numbered bz*ny+by; cell_start[cell_base + cell]
// is the global sorted position of the first cluster of the cell; the entry after the last cell of a bucket
// is the first cell of the next bucket (= bucket end), and one sentinel closes the table.
struct GridDesc {
  float y0, z0, inv_e;
  int32_t ny, nz;
  uint32_t cell_base;
  uint32_t lo, n;   // bucket range in the (sorted == input) CSR
};

struct DevParams {
  float area_y, area_z, link_dev2_max;
  float err2_y, err2_z, init_var_s, init_var_t, init_var_q, turn_var_scale;
  float max_sinphi, road_sigma, road_min, road_max;
  int32_t max_row_gap, min_chain_hits, min_tracklet_hits, min_track_hits;
  float cell_min, cell_max, clusters_per_cell;
  float b;                      // (float)(0.00299792458 * Bz)
  float tan_half_sector, z_min, z_max;
  int32_t n_rows, n_sectors, n_buckets;
  int32_t max_cells_per_bucket;
  int32_t any_dead;             // 1 if some row is dead (then the constructor fills the rows it steps over with -1)
};

// Device status / counter block (int64 slots), copied to pinned host memory at the end of a run.
enum Counter {
  CNT_ERROR = 0,        // sticky data-dependent error code (0 = ok)
  CNT_N_START = 1,      // start hits found (may exceed cap_tracklets)
  CNT_N_TRACKLETS = 2,  // accepted tracklets
  CNT_N_TL_HITS = 3,    // hits over accepted tracklets
  CNT_N_TRACKS = 4,     // tracks found (may exceed cap_tracks)
  CNT_N_TRK_CL = 5,     // track clusters (may exceed cap)
  CNT_N_CELLS = 6,
  CNT_WORK = 7,         // dynamic work counter of the constructor's up pass
  CNT_N_LONG = 8,       // seeds whose link chain is long enough to survive the chain fit (the constructor's work list)
  CNT_INF = 9,          // a count larger than any array: "scan everything" for the device-counted scan kernels
  CNT_WORK2 = 10,       // work counters of the two down-pass kernels of the constructor
  CNT_WORK3 = 11,
  CNT_WORK4 = 12,
  CNT_N_GAP = 13,       // seeds whose span has a gap row (the gap instance of the span pass)
  CNT_COUNT = 14
};

// Tracklet SoA in the workspace (capT = capacity in tracklets).
struct TrackletStore {
  int32_t* status;      // [capT]
  int32_t* nhits;       // [capT]
  int32_t* first_row;   // [capT]
  int32_t* last_row;    // [capT]
  int32_t* sector;      // [capT]
  float* x;             // [capT]
  float* par;           // [5][capT]
  float* cov;           // [15][capT]
  float* chi2;          // [capT]
  int32_t* rowhit;      // [capT][n_rows] sorted positions, valid for first_row..last_row only
  int64_t capT;
  int32_t n_rows;
};

__device__ __forceinline__ int cellCoord(float v, float v0, float inv_e, int n) {
  // monotone non-decreasing in v (fp32 subtract / multiply by a positive constant / floor / clamp all are),
  // which is what makes "cells of [lo,hi] enumerate a superset of the clusters in [lo,hi]" rigorous (R3).
  float f = floorf((v - v0) * inv_e);
  f = fminf(fmaxf(f, 0.0f), (float)(n - 1));   // NaN -> 0
  return (int)f;
}

// bucket of a sorted position: largest b with off[b] <= p (off has nb+1 entries, off[nb] = N > p)
__device__ __forceinline__ int bucketOf(const uint32_t* __restrict__ off, int nb, uint32_t p) {
  int lo = 0, hi = nb;   // invariant: off[lo] <= p < off[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (__ldg(off + mid) <= p) lo = mid; else hi = mid;
  }
  return lo;
}

__device__ __forceinline__ bool finitef(float v) { return (__float_as_uint(v) & 0x7f800000u) != 0x7f800000u; }

// Enumerate the clusters of one bucket inside the closed window [yc-wy, yc+wy] x [zc-wz, zc+wz].
// The grid gives a superset (whole cells, with slack for the rounding of the predicate's subtraction);
// the exact fp32 predicate of DESIGN.md O2/O4 decides.  f(pos, y, z) is called for every accepted cluster.
// One flat loop: an iteration either tests one candidate or advances to the next cell row, so that the lanes
// of a warp stay together whatever the lengths of their cell ranges are.
template <typename F>
__device__ __forceinline__ void forWindow(const GridDesc& G, const uint32_t* __restrict__ cell_start,
                                          const float2* __restrict__ syz, float yc, float zc, float wy, float wz, F&& f) {
  if (G.n == 0) return;
  const float sy = 1e-5f * (fabsf(yc) + wy) + 1e-6f;
  const float sz = 1e-5f * (fabsf(zc) + wz) + 1e-6f;
  const int by0 = cellCoord((yc - wy) - sy, G.y0, G.inv_e, G.ny);
  const int by1 = cellCoord((yc + wy) + sy, G.y0, G.inv_e, G.ny);
  int bz = cellCoord((zc - wz) - sz, G.z0, G.inv_e, G.nz);
  const int bz1 = cellCoord((zc + wz) + sz, G.z0, G.inv_e, G.nz);
  const uint32_t* cs = cell_start + G.cell_base + by0;
  const int span = by1 - by0 + 1;
  uint32_t k = __ldg(cs + bz * G.ny), kend = __ldg(cs + bz * G.ny + span);
  for (;;) {
    if (k < kend) {
      const float2 c = __ldg(syz + k);
      if (fabsf(c.x - yc) <= wy && fabsf(c.y - zc) <= wz) f(k, c.x, c.y);
      ++k;
    } else {
      if (++bz > bz1) break;
      k = __ldg(cs + bz * G.ny);
      kend = __ldg(cs + bz * G.ny + span);
    }
  }
}

}  // namespace tpc
