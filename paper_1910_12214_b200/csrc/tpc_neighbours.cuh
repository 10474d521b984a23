// tpc_neighbours.cuh -- a2 neighbour finder (O2; R2, R4..R7).
//
// For every cluster h on row r:  U = clusters of row up(r) with |y_u-y_h| <= area_y*dxu and |z_u-z_h| <= area_z*dxu,
// D likewise on row dn(r);  tyu=(y_u-y_h)*iu, tzu=(z_u-z_h)*iu, tyd=(y_h-y_d)*id, tzd=(z_h-z_d)*id;
// Dev(u,d) = (tyu-tyd)^2 + (tzu-tzd)^2;  best = argmin of (Dev, orig(u), orig(d));  link both iff Dev <= link_dev2_max.
//
// Organisation (one CTA = up to 128 consecutive sorted clusters of ONE (sector,row) bucket):
//   1. the clusters of a CTA are neighbours in z (the grid order is z-major), so all their up / down candidates
//      lie in two CONTIGUOUS ranges of the sorted array: both are staged in shared memory with coalesced loads;
//   2. each thread walks the grid cells of its own windows and keeps the 16-bit region indices of the clusters
//      that pass the exact predicate (its U and D lists);
//   3. the nU x nD pair loop is NOT run per cluster (nU*nD varies from 1 to >500 inside a warp): the (h,u)
//      combinations of the whole CTA become a flat item list and every lane takes items, looping over the D
//      list of the item's h -- lanes of a warp mostly share h, so the loop lengths agree and reads broadcast;
//   4. each thread reduces the results of its own items with the full lexicographic key.
// Anything that does not fit the fixed shared-memory budget (huge regions, > NF_LIST candidates in a window,
// > NF_ITEMS items) takes a per-thread slow path with the same predicate, arithmetic and key.
#pragma once
#include "tpc_common.cuh"

namespace tpc {

#ifndef NF_THREADS_
#define NF_THREADS_ 128
#endif
constexpr int NF_THREADS = NF_THREADS_;
#ifndef NF_REGION_
#define NF_REGION_ 640
#endif
constexpr int NF_REGION = NF_REGION_;     // staged candidates per side
#ifndef NF_LIST_
#define NF_LIST_ 32
#endif
#ifndef NF_ITEMS_
#define NF_ITEMS_ 512
#endif
constexpr int NF_LIST = NF_LIST_;  // window candidates kept per thread and side (<= 32: packed item code)
#ifndef NF_UB_
#define NF_UB_ 4
#endif
constexpr int NF_UB = NF_UB_;          // u's per item (register blocking of the pair loop)
constexpr int NF_ITEMS = NF_ITEMS_; // items per CTA and round
#ifndef NF_GUNROLL_
#define NF_GUNROLL_ 2
#endif
constexpr int NF_GUNROLL = NF_GUNROLL_;
#ifndef NF_DUNROLL_
#define NF_DUNROLL_ 2
#endif
constexpr int NF_DUNROLL = NF_DUNROLL_;   // unrolling of the D loop of the pair phase
constexpr int NF_ROWS = 6;         // cell rows of a window whose ranges are staged (more: slow path)

struct RowTables {
  const float* row_x;     // [R]
  const int16_t* up_row;  // [R] first live row among r+1, r+2 or -1 (R2); -1 for dead rows
  const int16_t* dn_row;  // [R]
  const uint8_t* dead;    // [R]
};

__device__ __forceinline__ void nfCpAsync8(void* smem, const void* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(sa), "l"(gmem) : "memory");
}

// region entry at a byte offset (the window lists hold 8 * index: 16 bits are enough, bit 15 stays free for the tie flag)
static_assert(NF_REGION * 8 <= 0x8000, "byte offsets of the region must fit 15 bits");
__device__ __forceinline__ float2 nfAt(const float2* reg, uint32_t byte_off) {
  return *reinterpret_cast<const float2*>(reinterpret_cast<const char*>(reg) + byte_off);
}

// lexicographic (Dev, orig(u), orig(d)) "is the new pair better" (R6)
__device__ __forceinline__ bool pairBetter(bool have, float dev, float best, uint32_t u, uint32_t d, uint32_t bu,
                                           uint32_t bd, const uint32_t* __restrict__ s2o) {
  if (!have || dev < best) return true;
  if (dev != best) return false;
  if (u != bu) return __ldg(s2o + u) < __ldg(s2o + bu);
  return __ldg(s2o + d) < __ldg(s2o + bd);
}

// per-thread reference path: nested enumeration of both windows straight from global memory
__device__ __noinline__ void neighbourSlow(uint32_t p, float2 h, const GridDesc& Gu, const GridDesc& Gd,
                                           const uint32_t* __restrict__ cell_start, const float2* __restrict__ syz,
                                           const uint32_t* __restrict__ s2o, float iu, float id, float wyu, float wzu,
                                           float wyd, float wzd, float dev_max, int32_t* __restrict__ lup,
                                           int32_t* __restrict__ ldn) {
  bool have = false;
  float best = 0.0f;
  uint32_t bu = 0, bd = 0;
  forWindow(Gu, cell_start, syz, h.x, h.y, wyu, wzu, [&](uint32_t u, float yu, float zu) {
    const float tyu = (yu - h.x) * iu, tzu = (zu - h.y) * iu;
    forWindow(Gd, cell_start, syz, h.x, h.y, wyd, wzd, [&](uint32_t d, float yd, float zd) {
      const float tyd = (h.x - yd) * id, tzd = (h.y - zd) * id;
      const float ey = tyu - tyd, ez = tzu - tzd;
      const float dev = ey * ey + ez * ez;
      if (pairBetter(have, dev, best, u, d, bu, bd, s2o)) { have = true; best = dev; bu = u; bd = d; }
    });
  });
  const bool link = have && best <= dev_max;
  lup[p] = link ? (int32_t)bu : -1;
  ldn[p] = link ? (int32_t)bd : -1;
}

// window walk over a region staged in shared memory: the cluster ranges of the window's cell rows come from the
// global cell table (all requested at once, kept as 16-bit region offsets in `rows`), the coordinates from `reg`
// (region index = sorted position - k0).  Appends the indices passing the predicate; returns their number, or
// NF_LIST + 1 when the window spans more than NF_ROWS cell rows (the caller then takes the slow path).
__device__ __forceinline__ int gatherWindow(const GridDesc& G, const uint32_t* __restrict__ cell_start, const float2* reg,
                                            uint32_t k0, float yc, float zc, float wy, float wz, uint16_t* list,
                                            ushort2* rows, int tid) {      // rows: the warp's own [NF_ROWS][32] slice
  const int lane = tid & 31;
  if (G.n == 0) return 0;
  const float sy = 1e-5f * (fabsf(yc) + wy) + 1e-6f;
  const float sz = 1e-5f * (fabsf(zc) + wz) + 1e-6f;
  const int by0 = cellCoord((yc - wy) - sy, G.y0, G.inv_e, G.ny);
  const int by1 = cellCoord((yc + wy) + sy, G.y0, G.inv_e, G.ny);
  const int bz0 = cellCoord((zc - wz) - sz, G.z0, G.inv_e, G.nz);
  const int nr = cellCoord((zc + wz) + sz, G.z0, G.inv_e, G.nz) - bz0 + 1;
  if (nr > NF_ROWS) return NF_LIST + 1;
  const uint32_t* cs = cell_start + G.cell_base + by0 + bz0 * G.ny;
  const int span = by1 - by0 + 1;
  uint32_t ra[NF_ROWS], rb[NF_ROWS];
#pragma unroll
  for (int r = 0; r < NF_ROWS; ++r) {
    const uint32_t* c = cs + (r < nr ? r : 0) * G.ny;
    ra[r] = __ldg(c); rb[r] = __ldg(c + span);
  }
  // the ranges are kept as BYTE offsets into the region (8 bytes per cluster; at most 8 * NF_REGION: 16 bits)
#pragma unroll
  for (int r = 0; r < NF_ROWS; ++r) rows[r * 32 + lane] = make_ushort2((uint16_t)((ra[r] - k0) << 3), (uint16_t)((rb[r] - k0) << 3));
  // The loop body is eight instructions per candidate: one shared load, one packed subtraction (FADD2: each half is the
  // IEEE c - centre, as c + (-centre)), two compares, the store of the byte offset to the slot the cursor points at (clamped
  // to the spare row NF_LIST: no branch), the cursor advanced by one row when the candidate passes.  The cursor is a
  // shared-memory ADDRESS (not a count times a stride plus a base: that was seven more instructions, r2e), the count comes
  // out of it at the end.
  const uint32_t l0 = (uint32_t)__cvta_generic_to_shared(list + tid);
  const uint32_t lmax = l0 + NF_LIST * NF_THREADS * (uint32_t)sizeof(uint16_t);
  uint32_t la = l0;
  const float2 nc = make_float2(-yc, -zc);
  for (int r = 0; r < nr; ++r) {
    const ushort2 v = rows[r * 32 + lane];
#pragma unroll NF_GUNROLL
    for (uint32_t k8 = v.x; k8 < v.y; k8 += 8) {
      const float2 d = __fadd2_rn(nfAt(reg, k8), nc);
      asm volatile("st.shared.u16 [%0], %1;" ::"r"(min(la, lmax)), "h"((uint16_t)k8) : "memory");
      // pass = |dy| <= wy && |dz| <= wz (false for NaN); the cursor moves on under that predicate: three instructions
      asm("{\n\t.reg .pred p;\n\t.reg .f32 a, b;\n\tabs.f32 a, %1;\n\tabs.f32 b, %2;\n\tsetp.le.f32 p, a, %3;\n\t"
          "setp.le.and.f32 p, b, %4, p;\n\t@p add.u32 %0, %0, %5;\n\t}"
          : "+r"(la)
          : "f"(d.x), "f"(d.y), "f"(wy), "f"(wz), "n"(NF_THREADS * (int)sizeof(uint16_t)));
    }
  }
  return (int)((la - l0) / (NF_THREADS * (uint32_t)sizeof(uint16_t)));
}

// thread per neighbour-finder CTA: its bucket (largest b with chunk_base[b] <= cta), so that the CTAs themselves start
// with one load instead of a dependent binary search by one thread while 127 wait
__global__ void __launch_bounds__(256) chunkFill(const uint32_t* __restrict__ chunk_base, int nb, int64_t max_chunks,
                                                 uint32_t* __restrict__ chunk_bucket, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= max_chunks || c >= __ldg(chunk_base + nb)) return;
  int lo = 0, hi = nb;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(chunk_base + mid) <= (uint32_t)c) lo = mid; else hi = mid;
  }
  chunk_bucket[c] = (uint32_t)lo;
}

// One warp per neighbour-finder CTA (chunk of NF_THREADS consecutive sorted clusters of one bucket), after chunkFill: the
// z extent of the chunk and from it the two CONTIGUOUS candidate ranges of the sorted array, [kD0, kD1) on the row below and
// [kU0, kU1) on the row above (all zero when the row has no row pair).  Inside neighbourFinder this was a block reduction
// and four dependent cell-table loads in front of the staging copies: three memory latencies per CTA before its first
// useful instruction (16 % of the kernel's stall samples sat in that prologue, profiles/r2e).  Here it is throughput
// work, and the CTA starts with two 16-byte loads: the ranges, and (first cluster, end of the bucket, bucket).
__global__ void __launch_bounds__(256) chunkRegions(const uint32_t* __restrict__ chunk_base,
                                                    const uint32_t* __restrict__ chunk_bucket, DevParams P, RowTables T,
                                                    const GridDesc* __restrict__ desc,
                                                    const uint32_t* __restrict__ cell_start,
                                                    const float2* __restrict__ syz, uint4* __restrict__ chunk_reg,
                                                    const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int nb = P.n_buckets;
  const uint32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;      // warp = chunk
  const int lane = threadIdx.x & 31;
  if (c >= __ldg(chunk_base + nb)) return;
  const int b = (int)__ldg(chunk_bucket + c);
  const GridDesc Gh = desc[b];
  const int r = b % P.n_rows;
  const int ru = T.up_row[r], rd = T.dn_row[r];
  const uint32_t p0 = Gh.lo + (c - __ldg(chunk_base + b)) * NF_THREADS, pend = Gh.lo + Gh.n;
  if (lane == 0) chunk_reg[2 * c + 1] = make_uint4(p0, pend, (uint32_t)b, 0u);
  if (ru < 0 || rd < 0) {
    if (lane == 0) chunk_reg[2 * c] = make_uint4(0u, 0u, 0u, 0u);
    return;
  }
  // the descriptors of the two neighbour rows are requested together with the clusters (one memory latency, not two)
  const GridDesc Gu = desc[b - r + ru], Gd = desc[b - r + rd];
  float zlo = 3.0e38f, zhi = -3.0e38f;
#pragma unroll
  for (int k = 0; k < NF_THREADS / 32; ++k) {
    const uint32_t p = p0 + k * 32 + lane;
    if (p < pend) { const float z = syz[p].y; zlo = fminf(zlo, z); zhi = fmaxf(zhi, z); }
  }
  for (int d = 16; d > 0; d >>= 1) {
    zlo = fminf(zlo, __shfl_xor_sync(0xffffffffu, zlo, d));
    zhi = fmaxf(zhi, __shfl_xor_sync(0xffffffffu, zhi, d));
  }
  if (lane != 0) return;
  const float xr = T.row_x[r];
  const float dxu = T.row_x[ru] - xr, dxd = xr - T.row_x[rd];
  const float wzu = P.area_z * dxu, wzd = P.area_z * dxd;
  uint32_t kD0 = 0, kD1 = 0, kU0 = 0, kU1 = 0;
  const float s = 1e-5f * (fmaxf(fabsf(zlo), fabsf(zhi)) + wzu + wzd) + 1e-6f;
  if (Gd.n) {
    const int a = cellCoord((zlo - wzd) - s, Gd.z0, Gd.inv_e, Gd.nz), e = cellCoord((zhi + wzd) + s, Gd.z0, Gd.inv_e, Gd.nz);
    kD0 = __ldg(cell_start + Gd.cell_base + a * Gd.ny);
    kD1 = __ldg(cell_start + Gd.cell_base + (e + 1) * Gd.ny);
  }
  if (Gu.n) {
    const int a = cellCoord((zlo - wzu) - s, Gu.z0, Gu.inv_e, Gu.nz), e = cellCoord((zhi + wzu) + s, Gu.z0, Gu.inv_e, Gu.nz);
    kU0 = __ldg(cell_start + Gu.cell_base + a * Gu.ny);
    kU1 = __ldg(cell_start + Gu.cell_base + (e + 1) * Gu.ny);
  }
  chunk_reg[2 * c] = make_uint4(kD0, kD1, kU0, kU1);
}

__global__ void __launch_bounds__(NF_THREADS) neighbourFinder(const uint32_t* __restrict__ chunk_base,
                                                              const uint32_t* __restrict__ chunk_bucket,
                                                              const uint4* __restrict__ chunk_reg, DevParams P, RowTables T,
                                                              const GridDesc* __restrict__ desc,
                                                              const uint32_t* __restrict__ cell_start,
                                                              const float2* __restrict__ syz,
                                                              const uint32_t* __restrict__ s2o, int32_t* __restrict__ lup,
                                                              int32_t* __restrict__ ldn, const int64_t* __restrict__ cnt) {
  __shared__ float2 sD[NF_REGION], sU[NF_REGION], sH[NF_THREADS];
  __shared__ uint16_t dl[(NF_LIST + 1) * NF_THREADS], ul[(NF_LIST + 1) * NF_THREADS];
  __shared__ uint16_t it[NF_ITEMS];
  __shared__ float it_dev[NF_ITEMS * NF_UB];
  __shared__ uint8_t snD[NF_THREADS], snU[NF_THREADS];
  // From the staging barrier on every warp works for itself: its 32 clusters, their lists, its own slice of the item
  // arrays (NF_WITEMS items), warp scans and __syncwarp -- no block barrier in the rounds (three per round and a block scan
  // before: a tenth of the kernel's stall samples, profiles/r2e).
  constexpr int NF_WITEMS = NF_ITEMS / (NF_THREADS / 32);
  static_assert(NF_WITEMS >= 32 / NF_UB + 1, "a cluster's items must fit a warp's slice");
  static_assert(sizeof(float) * NF_WITEMS * NF_UB >= sizeof(ushort2) * NF_ROWS * 32, "srow aliases the warp's slice of it_dev");
  if (cnt[CNT_ERROR] != 0) return;
  const int tid = threadIdx.x;
  const int lane = tid & 31, wbase = (tid >> 5) * NF_WITEMS;
  ushort2* srow = reinterpret_cast<ushort2*>(it_dev + wbase * NF_UB);   // cell-row ranges: only live while the lists are built
  const int nb = P.n_buckets;
  if (blockIdx.x >= __ldg(chunk_base + nb)) return;
  const uint4 kr = __ldg(chunk_reg + 2 * blockIdx.x), kq = __ldg(chunk_reg + 2 * blockIdx.x + 1);
  const int b = (int)kq.z;
  const uint32_t p = kq.x + tid;
  const bool valid = p < kq.y;
  const int r = b % P.n_rows;
  const int ru = T.up_row[r], rd = T.dn_row[r];
  if (ru < 0 || rd < 0) {   // no row pair (first / last rows, dead rows): no links (uniform branch)
    if (valid) { lup[p] = -1; ldn[p] = -1; }
    return;
  }
  const float xr = T.row_x[r];
  const float dxu = T.row_x[ru] - xr, dxd = xr - T.row_x[rd];
  const float iu = 1.0f / dxu, id = 1.0f / dxd;
  const float wyu = P.area_y * dxu, wzu = P.area_z * dxu;
  const float wyd = P.area_y * dxd, wzd = P.area_z * dxd;
  const GridDesc Gu = desc[b - r + ru], Gd = desc[b - r + rd];
  const float2 h = valid ? syz[p] : make_float2(0.0f, 0.0f);

  // ---- the contiguous candidate regions of the chunk: computed by chunkRegions ----
  const uint32_t kD0 = kr.x, kD1 = kr.y, kU0 = kr.z, kU1 = kr.w;
  if (kD1 - kD0 > NF_REGION || kU1 - kU0 > NF_REGION) {     // regions too large for shared memory (uniform branch)
    if (valid) neighbourSlow(p, h, Gu, Gd, cell_start, syz, s2o, iu, id, wyu, wzu, wyd, wzd, P.link_dev2_max, lup, ldn);
    return;
  }
  // both regions by asynchronous 8-byte copies: every load of the thread is in flight before the first one is waited for
  for (uint32_t i = tid; i < kD1 - kD0; i += NF_THREADS) nfCpAsync8(sD + i, syz + kD0 + i);
  for (uint32_t i = tid; i < kU1 - kU0; i += NF_THREADS) nfCpAsync8(sU + i, syz + kU0 + i);
  asm volatile("cp.async.wait_all;\n" ::: "memory");
  sH[tid] = h;
  __syncthreads();

  // ---- per-thread window lists ----
  int nD = 0, nU = 0;
  if (valid) {
    nD = gatherWindow(Gd, cell_start, sD, kD0, h.x, h.y, wyd, wzd, dl, srow, tid);
    if (nD > 0) nU = gatherWindow(Gu, cell_start, sU, kU0, h.x, h.y, wyu, wzu, ul, srow, tid);
  }
  const bool slow = nD > NF_LIST || nU > NF_LIST;
  snD[tid] = (uint8_t)min(nD, NF_LIST);
  snU[tid] = (uint8_t)min(nU, NF_LIST);
  bool pending = nD > 0 && nU > 0 && !slow;        // still has to put its nU items through the pair phase
  bool have = false, tied = false;
  float best = 0.0f;
  uint32_t bu = 0, bd = 0;
  // A warp's item list holds NF_WITEMS (h,u) items; warps with more run the pair phase in several rounds.
  __syncwarp();                                     // the lists and counts of the warp's clusters are written
  for (;;) {
    const uint32_t mine = pending ? (uint32_t)((nU + NF_UB - 1) / NF_UB) : 0u;     // items: groups of NF_UB u's
    const uint32_t inc = warpInclusiveScan(mine);
    if (__shfl_sync(0xffffffffu, inc, 31) == 0) break;      // uniform over the warp
    const uint32_t base = inc - mine;
    const bool now = pending && base + mine <= NF_WITEMS;   // the clusters that fit are a prefix: no holes in the list
    if (now)
      for (uint32_t a = 0; a < mine; ++a) it[wbase + base + a] = (uint16_t)(tid * 32 + a * NF_UB);
    const uint32_t Tn = __reduce_max_sync(0xffffffffu, now ? base + mine : 0u);    // end of the last cluster that fitted
    __syncwarp();
    // ---- pair phase: one item = (h, NF_UB consecutive u's of its list); loop over the D list of h.
    //      The down slopes are computed once per d and used for all u's of the item (register blocking).
    for (uint32_t iw = lane; iw < Tn; iw += 32) {
      const uint32_t i = wbase + iw;
      const uint32_t e = it[i];
      const int hl = e >> 5, a0 = e & 31;
      const float2 hh = sH[hl];
      const int nu = snU[hl];
      // The slopes are kept as (y, z) pairs and subtracted / squared with the packed fp32 instructions of sm_100
      // (FADD2 / FMUL2: each half is the IEEE round-to-nearest operation, so the result is bit-identical to the
      // scalar form; one issue slot for two operations).  ptxas contracts a packed mul that feeds a packed add into
      // FFMA2 even with --fmad=false and explicit .rn (measured), so that pattern is never
      // written: the differences of two slopes (products) are scalar adds, and only add -> mul and mul -> scalar add
      // chains are packed (tests/test_build_flags.py checks the SASS of the library for FFMA2).
      // The pair loop keeps only the MINIMUM of Dev over the D list of every (h, u) (one FMNMX per pair; the running
      // argmin and the tie flag were four instructions per pair, 93 pairs per cluster).  Which d it was is found
      // afterwards, by the cluster's own thread, for the winning u alone: the same arithmetic once more over its D list,
      // looking for the value (a second d with it = an exact tie, redone by neighbourSlow with the full key, R6).
      float2 tu[NF_UB];
      float bdev[NF_UB];
      const float2 iu2 = make_float2(iu, iu), id2 = make_float2(id, id), nh = make_float2(-hh.x, -hh.y);
#pragma unroll
      for (int q = 0; q < NF_UB; ++q) {
        const float2 uu = nfAt(sU, ul[min(a0 + q, nu - 1) * NF_THREADS + hl]);     // a short last group repeats its last u
        tu[q] = __fmul2_rn(__fadd2_rn(uu, nh), iu2);                         // ((y_u - y_h) * iu, (z_u - z_h) * iu)
        bdev[q] = __int_as_float(0x7f800000);
      }
      const int n = snD[hl];
#pragma unroll NF_DUNROLL
      for (int j = 0; j < n; ++j) {
        const uint32_t di = dl[j * NF_THREADS + hl];                         // byte offset of d in the region
        const float2 dd = nfAt(sD, di);
        const float2 ntd = __fmul2_rn(__fadd2_rn(dd, nh), id2);              // -(tyd, tzd): -((y_h - y_d) * id) exactly
#pragma unroll
        for (int q = 0; q < NF_UB; ++q) {
          const float2 e = make_float2(tu[q].x + ntd.x, tu[q].y + ntd.y);    // (tyu - tyd, tzu - tzd): scalar, see above
          const float2 m = __fmul2_rn(e, e);
          const float dev = m.x + m.y;
          // Window slopes are bounded by area_y/area_z, so dev is finite: +inf is a safe "none yet".
          bdev[q] = fminf(bdev[q], dev);
        }
      }
#pragma unroll
      for (int q = 0; q < NF_UB; ++q) it_dev[i * NF_UB + q] = bdev[q];
    }
    __syncwarp();
    // ---- per-cluster reduction over its own items, full key (Dev, orig u, orig d) ----
    if (now) {
      // branch-free: the minimum over the cluster's own u's; an exact tie between two u's only raises `tied` (the
      // cluster is then redone by neighbourSlow, R6)
      float bst = __int_as_float(0x7f800000);
      int ba = 0;
      for (int a = 0; a < nU; ++a) {
        const float dev = it_dev[(wbase + base) * NF_UB + a];
        tied = tied || dev == bst;
        const bool better = dev < bst;
        ba = better ? a : ba;
        bst = better ? dev : bst;
      }
      // the d of the winning u: Dev of (u*, d) recomputed with the pair loop's own operations, bit for bit
      const uint32_t ucode = ul[ba * NF_THREADS + tid];
      uint32_t bcode = 0, hits = 0;
      {
        const float2 iu2 = make_float2(iu, iu), id2 = make_float2(id, id), nh = make_float2(-h.x, -h.y);
        const float2 tu = __fmul2_rn(__fadd2_rn(nfAt(sU, ucode), nh), iu2);
        for (int j = nD - 1; j >= 0; --j) {           // downwards: the last match kept is the first of the list
          const uint32_t di = dl[j * NF_THREADS + tid];
          const float2 ntd = __fmul2_rn(__fadd2_rn(nfAt(sD, di), nh), id2);
          const float2 e = make_float2(tu.x + ntd.x, tu.y + ntd.y);
          const float2 m = __fmul2_rn(e, e);
          const bool eq = m.x + m.y == bst;
          bcode = eq ? di : bcode;
          hits += eq ? 1u : 0u;
        }
      }
      tied = tied || hits != 1u;                    // two d's at the minimum: a tie; none cannot happen (then: slow path)
      have = true; best = bst;                      // nU >= 1 here, and every dev is finite
      bu = kU0 + (ucode >> 3); bd = kD0 + (bcode >> 3);
      pending = false;
    }
    __syncwarp();                                   // the item arrays are rewritten in the next round
  }
  if (!valid) return;
  if (slow || tied) {
    neighbourSlow(p, h, Gu, Gd, cell_start, syz, s2o, iu, id, wyu, wzu, wyd, wzd, P.link_dev2_max, lup, ldn);
    return;
  }
  const bool link = have && best <= P.link_dev2_max;
  lup[p] = link ? (int32_t)bu : -1;
  ldn[p] = link ? (int32_t)bd : -1;
}

}  // namespace tpc
