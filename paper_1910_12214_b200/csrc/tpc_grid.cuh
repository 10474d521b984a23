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

// One CTA per (sector,row) bucket: counting sort of the bucket's clusters by grid cell, in shared memory.
//   pass 1  cell of every cluster, histogram by shared-memory atomics (coalesced loads of y and z);
//   pass 2  exclusive scan of the histogram (every thread scans a run of cells, one block scan joins the runs); the
//           bucket's slice of the global cell table is written once, coalesced;
//   pass 3  y, z read again (L2: the bucket was read a moment ago), slot = atomic cursor of the cell; (y,z) are scattered
//           into a stage in shared memory behind the histogram and written out as whole lines, then the input indices the
//           same way through the same stage (the slots wait in registers).  Scattered straight to global memory -- the
//           first form of this kernel, still the path of a bucket that does not fit the stage -- the two stores per
//           cluster were 1.0 ms of 1.35 ms: a warp's store went to 32 sectors.
// The bucket comes from blockIdx: no per-cluster search of row_offset, no global atomics, no memset of the cell table,
// no rank array (round 1: thread per cluster, a 13-step binary search and a global atomic each, twice: 2.4 ms on config 4).
// The in-cell order is the arrival order of the cursor atomics: free by R3.  A bucket whose cells do not fit the shared
// array (more than `smem_cells`) runs the same passes with its slice of the global table as the histogram and the
// arrival ranks kept in `rank`.  Histogram (up to 96 KB) + stage (8 bytes per cluster) = one CTA of 1024 threads per SM.
constexpr int GB_THREADS = 1024;
#ifndef GB_UNROLL_
#define GB_UNROLL_ 4
#endif
constexpr int GB_UNROLL = GB_UNROLL_;
#ifndef GB_STAGED
#define GB_STAGED 1
#endif
constexpr int GB_MAXC = 16;          // clusters per thread whose slots the staged scatter keeps in registers

__global__ void __launch_bounds__(GB_THREADS) gridBuild(const uint32_t* __restrict__ off, const float* __restrict__ y,
                                                        const float* __restrict__ z, int nb, const GridDesc* __restrict__ desc,
                                                        uint32_t* __restrict__ cell_start, uint32_t* __restrict__ rank,
                                                        float2* __restrict__ syz, uint32_t* __restrict__ s2o,
                                                        int64_t* __restrict__ cnt, int validate, uint32_t smem_cells,
                                                        uint32_t smem_bytes) {
  extern __shared__ uint32_t sh_hist[];
  __shared__ uint32_t sm[33];
  if (cnt[CNT_ERROR] != 0 && cnt[CNT_ERROR] != -6) return;      // bad offsets or too many cells (gridSetup); -6 is ours
  const int b = blockIdx.x;
  const int tid = threadIdx.x;
  const GridDesc g = desc[b];
  const uint32_t nc = (uint32_t)g.ny * (uint32_t)g.nz;
  uint32_t* table = cell_start + g.cell_base;
  const bool in_smem = nc <= smem_cells;
  uint32_t* hist = in_smem ? sh_hist : table;
  for (uint32_t c = tid; c < nc; c += GB_THREADS) hist[c] = 0u;
  if (b == nb - 1 && tid == 0) table[nc] = g.lo + g.n;            // the closing sentinel of the whole table
  __syncthreads();
  const uint32_t lo = g.lo, hi = g.lo + g.n;
  bool bad = false;
  // four clusters per thread and trip: eight independent loads in flight before the first atomic (two CTAs of 1024
  // threads per SM then keep 64 KB on the way, what the HBM latency asks for)
  for (uint32_t i0 = lo + tid; i0 < hi; i0 += GB_UNROLL * GB_THREADS) {
    float yy[GB_UNROLL], zz[GB_UNROLL];
#pragma unroll
    for (int u = 0; u < GB_UNROLL; ++u) {
      const uint32_t i = i0 + u * GB_THREADS;
      yy[u] = i < hi ? y[i] : 0.0f; zz[u] = i < hi ? z[i] : 0.0f;
    }
#pragma unroll
    for (int u = 0; u < GB_UNROLL; ++u) {
      const uint32_t i = i0 + u * GB_THREADS;
      if (i < hi) {
        bad = bad || !(finitef(yy[u]) && finitef(zz[u]));
        const int cell = cellCoord(zz[u], g.z0, g.inv_e, g.nz) * g.ny + cellCoord(yy[u], g.y0, g.inv_e, g.ny);
        const uint32_t r = atomicAdd(hist + cell, 1u);
        if (!in_smem) rank[i] = r;
      }
    }
  }
  if (validate && bad) cnt[CNT_ERROR] = -6;
  __syncthreads();
  // exclusive scan: thread t owns the cells [t * run, (t + 1) * run)
  const uint32_t run = (nc + GB_THREADS - 1) / GB_THREADS;
  const uint32_t c0 = min((uint32_t)tid * run, nc), c1 = min(c0 + run, nc);
  uint32_t sum = 0;
  for (uint32_t c = c0; c < c1; ++c) sum += hist[c];
  uint32_t total;
  uint32_t pre = lo + blockExclusiveScan(sum, sm, &total);        // global sorted position of the run's first cluster
  for (uint32_t c = c0; c < c1; ++c) { const uint32_t v = hist[c]; hist[c] = pre; pre += v; }
  __syncthreads();
  if (in_smem) {
    for (uint32_t c = tid; c < nc; c += GB_THREADS) table[c] = hist[c];
    __syncthreads();      // the cursors below overwrite the starts: every start must be copied out first
  }
#if GB_STAGED
  // Staged scatter (the usual case: the bucket's (y, z) fit shared memory behind the histogram and a thread holds at most
  // GB_MAXC clusters).  Scattered straight to global memory, the 8-byte and 4-byte stores of a warp go to 32 different
  // sectors each: measured, they were 1.0 ms of the kernel's 1.35 ms (0.64 ms without the (y, z) stores, 0.72 ms without the
  // index stores).  Here the slot of every cluster comes from the same cursor atomic, (y, z) are scattered inside shared
  // memory and written out as whole lines, then the input indices the same way through the same buffer; the slots wait in
  // registers in between.
  const uint32_t stage_off = (nc + 3u) & ~3u;      // words: the stage starts 16-byte aligned behind the histogram
  if (in_smem && g.n <= (uint32_t)(GB_MAXC * GB_THREADS) && (size_t)stage_off * 4 + (size_t)g.n * 8 <= smem_bytes) {
    float2* st = reinterpret_cast<float2*>(sh_hist + stage_off);
    uint32_t* si = reinterpret_cast<uint32_t*>(st);
    uint32_t slot[GB_MAXC];
#pragma unroll
    for (int k = 0; k < GB_MAXC; ++k) {
      const uint32_t i = lo + tid + k * GB_THREADS;
      slot[k] = 0xffffffffu;
      if (i < hi) {
        const float yy = y[i], zz = z[i];
        const int cell = cellCoord(zz, g.z0, g.inv_e, g.nz) * g.ny + cellCoord(yy, g.y0, g.inv_e, g.ny);
        const uint32_t q = atomicAdd(hist + cell, 1u) - lo;
        slot[k] = q;
        st[q] = make_float2(yy, zz);
      }
    }
    __syncthreads();
    for (uint32_t j = tid; j < g.n; j += GB_THREADS) syz[lo + j] = st[j];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < GB_MAXC; ++k)
      if (slot[k] != 0xffffffffu) si[slot[k]] = lo + tid + k * GB_THREADS;
    __syncthreads();
    for (uint32_t j = tid; j < g.n; j += GB_THREADS) s2o[lo + j] = si[j];
    return;
  }
#endif
  for (uint32_t i0 = lo + tid; i0 < hi; i0 += GB_UNROLL * GB_THREADS) {
    float yy[GB_UNROLL], zz[GB_UNROLL];
#pragma unroll
    for (int u = 0; u < GB_UNROLL; ++u) {
      const uint32_t i = i0 + u * GB_THREADS;
      yy[u] = i < hi ? y[i] : 0.0f; zz[u] = i < hi ? z[i] : 0.0f;
    }
#pragma unroll
    for (int u = 0; u < GB_UNROLL; ++u) {
      const uint32_t i = i0 + u * GB_THREADS;
      if (i < hi) {
        const int cell = cellCoord(zz[u], g.z0, g.inv_e, g.nz) * g.ny + cellCoord(yy[u], g.y0, g.inv_e, g.ny);
        const uint32_t pos = in_smem ? atomicAdd(hist + cell, 1u) : hist[cell] + rank[i];
        syz[pos] = make_float2(yy[u], zz[u]);
        s2o[pos] = i;
      }
    }
  }
}

}  // namespace tpc
