// tpc_links.cuh -- a2 neighbour finder, a3 cleaner + start-hit finder   (O2, O3; R4..R8).
//
// All link arrays inside the library hold SORTED positions (the grid's order); the original input index
// (sorted_to_orig) enters only where the method defines a result through it: tie-breaks (R6) and the order
// of the start-hit list (R8).
#pragma once
#include "tpc_common.cuh"

namespace tpc {

constexpr int NF_THREADS = 128;
constexpr int NF_STASH = 12;      // down candidates kept per thread in shared memory; more -> re-enumeration

struct RowTables {
  const float* row_x;     // [R]
  const int16_t* up_row;  // [R] first live row among r+1, r+2 or -1 (R2); -1 for dead rows
  const int16_t* dn_row;  // [R]
  const uint8_t* dead;    // [R]
};

// lexicographic (Dev, orig(u), orig(d)) "is the new pair better" (R6)
__device__ __forceinline__ bool pairBetter(bool have, float dev, float best, uint32_t u, uint32_t d, uint32_t bu,
                                           uint32_t bd, const uint32_t* __restrict__ s2o) {
  if (!have || dev < best) return true;
  if (dev != best) return false;
  if (u != bu) return __ldg(s2o + u) < __ldg(s2o + bu);
  return __ldg(s2o + d) < __ldg(s2o + bd);
}

// thread per cluster (sorted position p).  O2:
//   U = clusters of row up(r) with |y_u-y_h| <= area_y*dxu and |z_u-z_h| <= area_z*dxu, D likewise on dn(r);
//   slopes tyu=(y_u-y_h)*iu ... tyd=(y_h-y_d)*id; Dev = (tyu-tyd)^2 + (tzu-tzd)^2; argmin of (Dev, orig u, orig d);
//   link both iff Dev_best <= link_dev2_max.
// Three phases per thread, each a flat loop (SIMT efficiency): gather D slopes into shared memory, gather U
// slopes into shared memory, then one loop over the nU*nD pairs.  Windows holding more than NF_STASH
// candidates on a side take the re-enumerating slow path (same predicate, same arithmetic, same key).
__global__ void __launch_bounds__(NF_THREADS) neighbourFinder(const uint32_t* __restrict__ off, int64_t N, DevParams P,
                                                              RowTables T, const GridDesc* __restrict__ desc,
                                                              const uint32_t* __restrict__ cell_start,
                                                              const float2* __restrict__ syz,
                                                              const uint32_t* __restrict__ s2o, int32_t* __restrict__ lup,
                                                              int32_t* __restrict__ ldn, const int64_t* __restrict__ cnt) {
  __shared__ float d_ty[NF_STASH][NF_THREADS], d_tz[NF_STASH][NF_THREADS];
  __shared__ float u_ty[NF_STASH][NF_THREADS], u_tz[NF_STASH][NF_THREADS];
  __shared__ uint32_t d_pos[NF_STASH][NF_THREADS], u_pos[NF_STASH][NF_THREADS];
  __shared__ int blk_b[2];
  if (cnt[CNT_ERROR] != 0) return;
  const int tid = threadIdx.x;
  const int64_t p0 = (int64_t)blockIdx.x * NF_THREADS;
  if (tid < 2) {   // buckets of the first and last cluster of the block: usually the same one
    const int64_t q = tid == 0 ? p0 : min(p0 + NF_THREADS, N) - 1;
    blk_b[tid] = bucketOf(off, P.n_buckets, (uint32_t)q);
  }
  __syncthreads();
  const int64_t p64 = p0 + tid;
  if (p64 >= N) return;
  const uint32_t p = (uint32_t)p64;
  const int b = blk_b[0] == blk_b[1] ? blk_b[0] : bucketOf(off, P.n_buckets, p);
  const int r = b % P.n_rows;
  const int ru = T.up_row[r], rd = T.dn_row[r];
  int32_t out_u = -1, out_d = -1;
  if (ru >= 0 && rd >= 0) {
    const float2 h = syz[p];
    const float xr = T.row_x[r];
    const float dxu = T.row_x[ru] - xr, dxd = xr - T.row_x[rd];
    const float iu = 1.0f / dxu, id = 1.0f / dxd;
    const float wyu = P.area_y * dxu, wzu = P.area_z * dxu;
    const float wyd = P.area_y * dxd, wzd = P.area_z * dxd;
    const GridDesc Gu = desc[b - r + ru], Gd = desc[b - r + rd];
    int nD = 0, nU = 0;
    forWindow(Gd, cell_start, syz, h.x, h.y, wyd, wzd, [&](uint32_t k, float yd, float zd) {
      if (nD < NF_STASH) { d_ty[nD][tid] = (h.x - yd) * id; d_tz[nD][tid] = (h.y - zd) * id; d_pos[nD][tid] = k; }
      ++nD;
    });
    if (nD > 0)
      forWindow(Gu, cell_start, syz, h.x, h.y, wyu, wzu, [&](uint32_t k, float yu, float zu) {
        if (nU < NF_STASH) { u_ty[nU][tid] = (yu - h.x) * iu; u_tz[nU][tid] = (zu - h.y) * iu; u_pos[nU][tid] = k; }
        ++nU;
      });
    bool have = false;
    float best = 0.0f;
    uint32_t bu = 0, bd = 0;
    if (nD <= NF_STASH && nU <= NF_STASH) {
      const int nP = nU * nD;
      int a = 0, c = 0;
      for (int i = 0; i < nP; ++i) {
        const float ey = u_ty[a][tid] - d_ty[c][tid], ez = u_tz[a][tid] - d_tz[c][tid];
        const float dev = ey * ey + ez * ez;
        if (!have || dev <= best) {
          const uint32_t u = u_pos[a][tid], d = d_pos[c][tid];
          if (pairBetter(have, dev, best, u, d, bu, bd, s2o)) { have = true; best = dev; bu = u; bd = d; }
        }
        if (++c == nD) { c = 0; ++a; }
      }
    } else if (nD > 0 && nU > 0) {   // a stash overflowed: enumerate both windows again, nested
      forWindow(Gu, cell_start, syz, h.x, h.y, wyu, wzu, [&](uint32_t u, float yu, float zu) {
        const float tyu = (yu - h.x) * iu, tzu = (zu - h.y) * iu;
        forWindow(Gd, cell_start, syz, h.x, h.y, wyd, wzd, [&](uint32_t d, float yd, float zd) {
          const float tyd = (h.x - yd) * id, tzd = (h.y - zd) * id;
          const float ey = tyu - tyd, ez = tzu - tzd;
          const float dev = ey * ey + ez * ez;
          if (pairBetter(have, dev, best, u, d, bu, bd, s2o)) { have = true; best = dev; bu = u; bd = d; }
        });
      });
    }
    if (have && best <= P.link_dev2_max) { out_u = (int32_t)bu; out_d = (int32_t)bd; }
  }
  lup[p] = out_u;
  ldn[p] = out_d;
}

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
