// tpc_grid.cuh -- a1: per (sector,row) cluster grid by counting sort over (y,z)   (O1, R3).
//
// The grid never decides a result (R3): every search applies the exact fp32 window predicate to a superset
// that the cells enumerate; cell size, in-cell order and clamping are free.  In-cell order here is the
// arrival order of an atomic counter, i.e. not reproducible -- all tie-breaks downstream use the ORIGINAL
// input index (sorted_to_orig), never the sorted position.
#pragma once
#include "tpc_common.cuh"

namespace tpc {

// One block.  Validates row_offset, sizes every bucket's grid and lays the cell tables out back to back.
__global__ void __launch_bounds__(1024) gridSetup(const uint32_t* __restrict__ off, int64_t N, DevParams P,
                                                  const float* __restrict__ row_x, GridDesc* __restrict__ desc,
                                                  uint32_t* __restrict__ chunk_base, int chunk, int64_t* __restrict__ cnt,
                                                  int64_t cap_cells) {
  __shared__ uint32_t sm[33];
  __shared__ int bad;
  const int nb = P.n_buckets;
  if (threadIdx.x == 0) { bad = (off[0] != 0u) || ((int64_t)off[nb] != N); cnt[CNT_INF] = (int64_t)1 << 62; }
  __syncthreads();
  for (int b = threadIdx.x; b < nb; b += blockDim.x)
    if (off[b + 1] < off[b]) bad = 1;
  __syncthreads();
  if (bad) {
    for (int b = threadIdx.x; b < nb; b += blockDim.x) { desc[b] = GridDesc{0.f, 0.f, 1.f, 1, 1, 0u, 0u, 0u}; chunk_base[b] = 0; }
    if (threadIdx.x == 0) { cnt[CNT_ERROR] = -2; cnt[CNT_N_CELLS] = 0; chunk_base[nb] = 0; }
    return;
  }
  uint32_t carry = 0, ccarry = 0;      // running cell / chunk totals
  const float Wz = P.z_max - P.z_min;
  for (int base = 0; base < nb; base += blockDim.x) {
    const int b = base + threadIdx.x;
    GridDesc g{0.f, 0.f, 1.f, 1, 1, 0u, 0u, 0u};
    uint32_t nc = 0, nch = 0;
    if (b < nb) {
      const int r = b % P.n_rows;
      const uint32_t lo = off[b], n = off[b + 1] - lo;
      const float hw = row_x[r] * P.tan_half_sector;
      const float Wy = 2.0f * hw;
      float e = n > 0 ? sqrtf(Wy * Wz * P.clusters_per_cell / (float)n) : P.cell_max;
      e = fminf(fmaxf(e, P.cell_min), P.cell_max);
      int ny, nz;
      for (;;) {
        ny = max(1, (int)ceilf(Wy / e));
        nz = max(1, (int)ceilf(Wz / e));
        if ((int64_t)ny * nz <= P.max_cells_per_bucket) break;
        e *= 1.25f;
      }
      g.y0 = -hw; g.z0 = P.z_min; g.inv_e = 1.0f / e; g.ny = ny; g.nz = nz; g.lo = lo; g.n = n;
      nc = (uint32_t)(ny * nz);
      nch = (n + chunk - 1) / chunk;      // CTAs of the neighbour finder: `chunk` clusters of one bucket each
    }
    uint32_t total;
    const uint32_t ex = blockExclusiveScan(nc, sm, &total);
    if (b < nb) { g.cell_base = carry + ex; desc[b] = g; }
    carry += total;
    const uint32_t cex = blockExclusiveScan(nch, sm, &total);
    if (b < nb) chunk_base[b] = ccarry + cex;
    ccarry += total;
  }
  if (threadIdx.x == 0) {
    chunk_base[nb] = ccarry;
    cnt[CNT_N_CELLS] = carry;
    if ((int64_t)carry > cap_cells) cnt[CNT_ERROR] = -3;
  }
}

// thread per cluster: cell of the cluster, rank inside the cell (arrival order), histogram in cell_cnt.
__global__ void __launch_bounds__(256) gridCount(const uint32_t* __restrict__ off, const float* __restrict__ y,
                                                 const float* __restrict__ z, int64_t N, int nb,
                                                 const GridDesc* __restrict__ desc, uint32_t* __restrict__ cell_cnt,
                                                 uint32_t* __restrict__ rank, int64_t* __restrict__ cnt, int validate) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int b = bucketOf(off, nb, (uint32_t)i);
  const GridDesc g = desc[b];
  const float yy = y[i], zz = z[i];
  if (validate && !(finitef(yy) && finitef(zz))) cnt[CNT_ERROR] = -6;
  const int cell = cellCoord(zz, g.z0, g.inv_e, g.nz) * g.ny + cellCoord(yy, g.y0, g.inv_e, g.ny);
  rank[i] = atomicAdd(cell_cnt + g.cell_base + cell, 1u);
}

// thread per cluster: sorted position = cell_start[cell] + rank; scatter (y,z) and the original index.
__global__ void __launch_bounds__(256) gridScatter(const uint32_t* __restrict__ off, const float* __restrict__ y,
                                                   const float* __restrict__ z, int64_t N, int nb,
                                                   const GridDesc* __restrict__ desc,
                                                   const uint32_t* __restrict__ cell_start,
                                                   const uint32_t* __restrict__ rank, float2* __restrict__ syz,
                                                   uint32_t* __restrict__ s2o, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int b = bucketOf(off, nb, (uint32_t)i);
  const GridDesc g = desc[b];
  const float yy = y[i], zz = z[i];
  const int cell = cellCoord(zz, g.z0, g.inv_e, g.nz) * g.ny + cellCoord(yy, g.y0, g.inv_e, g.ny);
  const uint32_t pos = cell_start[g.cell_base + cell] + rank[i];
  syz[pos] = make_float2(yy, zz);
  s2o[pos] = (uint32_t)i;
}

}  // namespace tpc
