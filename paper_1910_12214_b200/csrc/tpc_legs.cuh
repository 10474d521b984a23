// tpc_legs.cuh -- a10: optional pairs of track ends that are the two sides of a looper's outer turn (DESIGN.md section 3
// "O10", readings R40..R43; rest of NEXT-1 of SURVEY.md 8(f); loopers are found as several legs).
//
// A refitted track whose outer state is steep is a leg end.  Two leg ends with opposite inclinations, on the same side,
// at most leg_max_sectors sectors and leg_max_row_diff rows apart are compared in the frame halfway between their
// sectors, turned by 90 degrees -- the symmetry axis of the turn: the lower id is rotated by alpha = d*10 + sg*90 degrees
// and propagated (eight steps, R43) to the plane of the other, which is rotated by -alpha and mirrored; diagonal chi2.
// partner(k) = the compared end of minimal (chi2, id), kept when reciprocal.
//
// Organisation: the leg ends are bucketed by (sector, last row); one thread per leg end visits the buckets of the
// sectors it moves towards and of the rows around its own last row.  Every pair is evaluated by both of its ends with
// the same operands in the same order, so both see the same chi2 and no atomics are needed; a last pass keeps the
// reciprocal choices.
#pragma once
#include "tpc_kalman.cuh"
#include "tpc_merge.cuh"

namespace tpc {

constexpr int LEG_MAX_SECTORS = 8;          // d = 9 and d = -9 would be the same sector
constexpr int LEG_ANGLES = 2 * LEG_MAX_SECTORS + 2;

struct LegParams {
  float min_sinphi, chi2_max;
  int32_t max_sectors, max_row_diff;
  // (float)cos / sin of alpha = d*10 + sg*90 degrees and of -alpha, index d + LEG_MAX_SECTORS + (sg > 0)
  float ca[LEG_ANGLES], sa[LEG_ANGLES], cb[LEG_ANGLES], sb[LEG_ANGLES];
};
struct LegIn {
  int64_t cap;
  const int32_t *status, *sector, *last_row;
  const float *x_out, *par_out, *cov_out;
};
struct LegOut {
  int32_t* partner;
  float* chi2;
};

__device__ __forceinline__ bool legIsEnd(const LegIn& in, int64_t k, const LegParams& L) {
  return in.status[k] == 1 && !(fabsf(in.par_out[2 * in.cap + k]) < L.min_sinphi);
}

// per track: clear the outputs, count the leg ends per (sector, last row)
__global__ void __launch_bounds__(256) legCount(LegIn in, LegOut out, DevParams P, LegParams L, uint32_t* __restrict__ bucket_cnt,
                                                int32_t* __restrict__ best, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap) return;
  out.partner[k] = -1; out.chi2[k] = 0.0f; best[k] = -1;
  if (legIsEnd(in, k, L)) atomicAdd(bucket_cnt + in.sector[k] * P.n_rows + in.last_row[k], 1u);
}

// per leg end: its slot in the bucket list (the order inside a bucket is arbitrary: the argmin breaks ties by id)
__global__ void __launch_bounds__(256) legFill(LegIn in, DevParams P, LegParams L, const uint32_t* __restrict__ bucket_start,
                                               uint32_t* __restrict__ bucket_fill, uint32_t* __restrict__ list,
                                               const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap || !legIsEnd(in, k, L)) return;
  const int b = in.sector[k] * P.n_rows + in.last_row[k];
  list[bucket_start[b] + atomicAdd(bucket_fill + b, 1u)] = (uint32_t)k;
}

// O10 Mirror: frame turned by 180 degrees, helix walked backwards; C <- J C J^T, J = diag(-1, +1, +1, -1, -1)
__device__ __forceinline__ void kfMirror(KFState& S) {
  S.x = -S.x; S.y = -S.y; S.t = -S.t; S.q = -S.q;
  S.c10 = -S.c10; S.c20 = -S.c20; S.c31 = -S.c31; S.c32 = -S.c32; S.c41 = -S.c41; S.c42 = -S.c42;
}

// O10 LegMatch(a, b, d): a = the lower id; false when refused
__device__ __forceinline__ bool legMatchPair(KFState A, KFState B, int d, const DevParams& P, const LegParams& L, float& chi2) {
  const int ia = d + LEG_MAX_SECTORS + (A.s > 0.0f ? 1 : 0);
  if (!kfRotate(A, L.ca[ia], L.sa[ia], P)) return false;
  if (!kfRotate(B, L.cb[ia], L.sb[ia], P)) return false;
  kfMirror(B);
  const float x0 = A.x, step = (B.x - A.x) * 0.125f;
#pragma unroll 1
  for (int i = 1; i <= 8; ++i)
    if (!kfPropagate(A, i < 8 ? x0 + (float)i * step : B.x, P, [](float, float, float, float) {})) return false;
  const float pa[5] = {A.y, A.z, A.s, A.t, A.q}, pb[5] = {B.y, B.z, B.s, B.t, B.q};
  const float va[5] = {A.c00, A.c11, A.c22, A.c33, A.c44}, vb[5] = {B.c00, B.c11, B.c22, B.c33, B.c44};
  float sum = 0.0f;
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    const float den = va[i] + vb[i];
    if (!(den > 0.0f)) return false;
    const float dd = pa[i] - pb[i];
    sum = sum + (dd * dd) / den;
  }
  if (!(sum <= L.chi2_max)) return false;
  chi2 = sum;
  return true;
}

// one thread per leg end a: the compared end of minimal (chi2, id)
__global__ void __launch_bounds__(128) legMatch(LegIn in, DevParams P, LegParams L, const uint32_t* __restrict__ bucket_start,
                                                const uint32_t* __restrict__ list, int32_t* __restrict__ best,
                                                float* __restrict__ best_chi, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= cnt[CNT_N_TRACKS] || a >= in.cap || !legIsEnd(in, a, L)) return;
  const int64_t cap = in.cap;
  const int R = P.n_rows;
  const KFState A0 = mergeLoad(a, cap, in.x_out, in.par_out, in.cov_out);
  const int sec = in.sector[a], la = in.last_row[a];
  const int sg = A0.s > 0.0f ? 1 : -1;
  const int side = sec / 18, j = sec - side * 18;
  const int r_lo = max(0, la - L.max_row_diff), r_hi = min(R - 1, la + L.max_row_diff);
  int32_t bb = -1;
  float bchi = 0.0f;
  const int dmax = P.n_sectors == 36 ? L.max_sectors : 0;
  for (int dd = 0; dd <= dmax; ++dd) {
    const int d = sg * dd;                                   // a moves towards the sectors on this side of it
    const int sb = dd == 0 ? sec : side * 18 + (j + d + 18) % 18;
    const uint32_t* bs = bucket_start + sb * R;
    for (uint32_t i = bs[r_lo]; i < bs[r_hi + 1]; ++i) {       // the buckets of consecutive rows are contiguous
      const int64_t b = list[i];
      if (b == a) continue;
      if (!(A0.s * in.par_out[2 * cap + b] < 0.0f)) continue;  // opposite inclinations
      const KFState B0 = mergeLoad(b, cap, in.x_out, in.par_out, in.cov_out);
      float c2;
      const bool ok = a < b ? legMatchPair(A0, B0, d, P, L, c2) : legMatchPair(B0, A0, -d, P, L, c2);
      if (!ok) continue;
      if (bb < 0 || c2 < bchi || (c2 == bchi && (int32_t)b < bb)) { bb = (int32_t)b; bchi = c2; }
    }
  }
  best[a] = bb; best_chi[a] = bchi;
}

// a pair is kept when each is the other's choice (R42)
__global__ void __launch_bounds__(256) legLink(LegIn in, LegOut out, const int32_t* __restrict__ best,
                                               const float* __restrict__ best_chi, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap) return;
  const int32_t o = best[k];
  if (o >= 0 && best[o] == (int32_t)k) { out.partner[k] = o; out.chi2[k] = best_chi[k]; }
}

}  // namespace tpc
