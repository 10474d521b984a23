// tpc_legs.cuh -- a10: optional pairs of track ends that are the two sides of a looper's outer turn (DESIGN.md section 3
// "O10", readings R40..R43; rest of NEXT-1 of SURVEY.md 8(f); loopers are found as several legs).
//
// A refitted track whose outer state is steep is a leg end.  Two leg ends with opposite inclinations, on the same side,
// at most leg_max_sectors sectors and leg_max_row_diff rows apart are compared in the frame halfway between their
// sectors, turned by 90 degrees -- the symmetry axis of the turn: the lower id is rotated by alpha = d*10 + sg*90 degrees
// and propagated (eight steps, R43) to the plane of the other, which is rotated by -alpha and mirrored; diagonal chi2.
// partner(k) = the compared end of minimal (chi2, id), kept when reciprocal.
//
// Organisation: the leg ends are bucketed by (sector, sign of sin phi, last row, bin of the dip t); one thread per leg
// end visits the buckets of the sectors it moves towards, of the opposite inclination, of the rows around its own last
// row and of the dip bins that can hold a partner: the dip term of the chi2 needs no transport (see legMatch), the terms
// are non-negative, and the window uses the largest dip variance of the (sector, sign, row) plus rounding slack, so it
// is a superset of every admissible partner -- no result changes (same argument as R3 and as the merger's bins).
// Every pair is evaluated by both of its ends with the same operands in the same order, so both see the same chi2 and
// no atomics are needed; a last pass keeps the reciprocal choices.
#pragma once
#include "tpc_kalman.cuh"
#include "tpc_merge.cuh"

namespace tpc {

constexpr int LEG_MAX_SECTORS = 8;          // d = 9 and d = -9 would be the same sector
constexpr int LEG_ANGLES = 2 * LEG_MAX_SECTORS + 2;
constexpr int LEG_NTB = 64;                 // dip bins over [-LEG_TMAX, LEG_TMAX] (clamped outside)
constexpr float LEG_TMAX = 2.0f;
constexpr float LEG_VWIDE = 2e-5f;          // ends with a larger dip variance go to one extra bin that is always visited,
constexpr int LEG_BINS = LEG_NTB + 1;       // so that a few badly measured dips do not widen everybody's window

// (sector, sign, row) index and the dip bin inside it
__device__ __forceinline__ int legRowKey(int sector, bool positive, int row, int R) { return (sector * 2 + (positive ? 1 : 0)) * R + row; }
__device__ __forceinline__ int legDipBin(float t) { return cellCoord(t, -LEG_TMAX, (float)LEG_NTB / (2.0f * LEG_TMAX), LEG_NTB); }
__device__ __forceinline__ int legBin(float t, float var_t) { return var_t <= LEG_VWIDE ? legDipBin(t) : LEG_NTB; }

struct LegParams {
  float min_sinphi, chi2_max, max_centre_dist;
  int32_t max_sectors, max_row_diff;
  // (float)cos / sin of alpha = d*10 + sg*90 degrees and of -alpha, index d + LEG_MAX_SECTORS + (sg > 0)
  float ca[LEG_ANGLES], sa[LEG_ANGLES], cb[LEG_ANGLES], sb[LEG_ANGLES];
  float cd[2 * LEG_MAX_SECTORS + 1], sd[2 * LEG_MAX_SECTORS + 1];   // (float)cos / sin of d*20 degrees, index d + LEG_MAX_SECTORS
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

// per track: clear the outputs, count the leg ends per bucket, largest dip variance per (sector, sign, row)
__global__ void __launch_bounds__(256) legCount(LegIn in, LegOut out, DevParams P, LegParams L, uint32_t* __restrict__ bucket_cnt,
                                                uint32_t* __restrict__ max_var, int32_t* __restrict__ best,
                                                const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap) return;
  out.partner[k] = -1; out.chi2[k] = 0.0f; best[k] = -1;
  if (legIsEnd(in, k, L)) {
    const int sr = legRowKey(in.sector[k], in.par_out[2 * in.cap + k] > 0.0f, in.last_row[k], P.n_rows);
    const float vt = in.cov_out[9 * in.cap + k];
    atomicAdd(bucket_cnt + sr * LEG_BINS + legBin(in.par_out[3 * in.cap + k], vt), 1u);
    if (vt <= LEG_VWIDE) atomicMax(max_var + sr, __float_as_uint(vt));     // positive floats order like their bit patterns
  }
}

// per leg end: its slot in the bucket list (the order inside a bucket is arbitrary: the argmin breaks ties by id)
__global__ void __launch_bounds__(256) legFill(LegIn in, DevParams P, LegParams L, const uint32_t* __restrict__ bucket_start,
                                               uint32_t* __restrict__ bucket_fill, uint32_t* __restrict__ list,
                                               float4* __restrict__ rec, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap || !legIsEnd(in, k, L)) return;
  const int b = legRowKey(in.sector[k], in.par_out[2 * in.cap + k] > 0.0f, in.last_row[k], P.n_rows) * LEG_BINS +
                legBin(in.par_out[3 * in.cap + k], in.cov_out[9 * in.cap + k]);
  const uint32_t slot = bucket_start[b] + atomicAdd(bucket_fill + b, 1u);
  list[slot] = (uint32_t)k;
  // what the cheap tests of legMatch read, in list order: the candidates of a lane are a few contiguous runs
  rec[slot] = make_float4(in.par_out[3 * in.cap + k], in.par_out[4 * in.cap + k], in.cov_out[9 * in.cap + k], in.cov_out[14 * in.cap + k]);
}

// O10 Mirror: frame turned by 180 degrees, helix walked backwards; C <- J C J^T, J = diag(-1, +1, +1, -1, -1)
__device__ __forceinline__ void kfMirror(KFState& S) {
  S.x = -S.x; S.y = -S.y; S.t = -S.t; S.q = -S.q;
  S.c10 = -S.c10; S.c20 = -S.c20; S.c31 = -S.c31; S.c32 = -S.c32; S.c41 = -S.c41; S.c42 = -S.c42;
}

// O10 LegMatch(a, b, d) after its first step (legCentresClose): a = the lower id; false when refused
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

// R44, the first step of LegMatch(a, b, d): the circle centres of the two outer states, each in its own frame (b's is
// turned by d * 20 degrees), lie within max_centre_dist
__device__ __forceinline__ bool legCentresClose(float xa, float ya, float sa, float qa, float xb, float yb, float sb, float qb,
                                                int d, const DevParams& P, const LegParams& L) {
  const float ka = qa * P.b, kb = qb * P.b;
  const float xca = xa - sa / ka, yca = ya + sqrtf(1.0f - sa * sa) / ka;
  const float xcb = xb - sb / kb, ycb = yb + sqrtf(1.0f - sb * sb) / kb;
  const float cd = L.cd[d + LEG_MAX_SECTORS], sd = L.sd[d + LEG_MAX_SECTORS];
  const float ex = (xcb * cd - ycb * sd) - xca, ey = (xcb * sd + ycb * cd) - yca;
  return ex * ex + ey * ey <= L.max_centre_dist * L.max_centre_dist;
}

// one thread per leg end a: the compared end of minimal (chi2, id)
__global__ void __launch_bounds__(128) legMatch(LegIn in, DevParams P, LegParams L, const uint32_t* __restrict__ bucket_start,
                                                const uint32_t* __restrict__ max_var, const uint32_t* __restrict__ list,
                                                const float4* __restrict__ rec, int32_t* __restrict__ best,
                                                float* __restrict__ best_chi,
                                                const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  // the leg ends are taken in list order: the lanes of a warp hold ends of one (sector, sign, row, dip bin) or of its
  // neighbours, so they walk nearly the same runs of candidates
  const int64_t slot = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int R = P.n_rows;
  // Lanes without an end stay in the loops (predicated off): the row loop has the same trip count for every lane and
  // reconverges at __syncwarp().
  const bool live = slot < bucket_start[(int64_t)P.n_buckets * 2 * LEG_BINS];
  const int64_t a = live ? list[slot] : 0;
  const int64_t cap = in.cap;
  KFState A0{};
  if (live) A0 = mergeLoad(a, cap, in.x_out, in.par_out, in.cov_out);
  const int sec = live ? in.sector[a] : 0, la = live ? in.last_row[a] : 0;
  const int sg = A0.s > 0.0f ? 1 : -1;
  const int side = sec / 18, j = sec - side * 18;
  const int r_lo = max(0, la - L.max_row_diff), r_hi = min(R - 1, la + L.max_row_diff);
  int32_t bb = -1;
  float bchi = 0.0f;
  const int dmax = P.n_sectors == 36 ? L.max_sectors : 0;
  for (int dd = 0; dd <= dmax; ++dd) {
    const int d = sg * dd;                                     // a moves towards the sectors on this side of it
    const int sb = dd == 0 ? sec : side * 18 + (j + d + 18) % 18;
    for (int it = 0; it <= 2 * L.max_row_diff; ++it) {
      __syncwarp();
      const int r = la - L.max_row_diff + it;
      if (!(live && r >= r_lo && r <= r_hi)) continue;
      const int sr = legRowKey(sb, sg < 0, r, R);              // the other inclination
      const uint32_t* bs = bucket_start + sr * LEG_BINS;
      // dip bins that can hold a partner: |t_a + t_b| <= sqrt(chi2_max * (C33_a + max C33_b)), with slack; a window
      // that is not >= 0 means no positive denominator is possible among the binned ends
      const float w = sqrtf(L.chi2_max * (A0.c33 + __uint_as_float(max_var[sr]))) * 1.0001f + 1e-6f;
      const bool any = w >= 0.0f;
      const uint32_t j0 = bs[LEG_NTB], j1 = bs[LEG_BINS];      // the ends with a wide dip variance: always visited
      const uint32_t i0 = any ? bs[legDipBin(-A0.t - w)] : j0, i1 = any ? bs[legDipBin(-A0.t + w) + 1] : j0;
      for (uint32_t ii = i0; ii < i1 + (j1 - j0); ++ii) {
        const uint32_t i = ii < i1 ? ii : j0 + (ii - i1);
        // The dip and curvature terms of the chi2 need no transport: Rotate and Propagate leave t, q, C33 and C44 as
        // they are and Mirror only changes the signs, so these are the very values LegMatch adds at the end; the terms
        // are non-negative and rounding is monotone, so one of them above the cut means the sum is above it.
        const float4 rc = __ldg(rec + i);                      // t, q, C33, C44 of the candidate
        const float q_b = rc.y;
        const float dt = A0.t + rc.x, dq = A0.q + q_b;
        const float t3 = (dt * dt) / (A0.c33 + rc.z), t4 = (dq * dq) / (A0.c44 + rc.w);
        if (t3 > L.chi2_max || t4 > L.chi2_max) continue;
        const int64_t b = list[i];
        if (b == a) continue;
        const float s_b = in.par_out[2 * cap + b];
        if (!(A0.s * s_b < 0.0f)) continue;                    // opposite inclinations (sin phi = 0 is in the negative key)
        const float x_b = in.x_out[b], y_b = in.par_out[b];
        if (!(a < b ? legCentresClose(A0.x, A0.y, A0.s, A0.q, x_b, y_b, s_b, q_b, d, P, L)
                    : legCentresClose(x_b, y_b, s_b, q_b, A0.x, A0.y, A0.s, A0.q, -d, P, L))) continue;
        const KFState B0 = mergeLoad(b, cap, in.x_out, in.par_out, in.cov_out);
        float c2;
        const bool ok = a < b ? legMatchPair(A0, B0, d, P, L, c2) : legMatchPair(B0, A0, -d, P, L, c2);
        if (!ok) continue;
        if (bb < 0 || c2 < bchi || (c2 == bchi && (int32_t)b < bb)) { bb = (int32_t)b; bchi = c2; }
      }
    }
  }
  if (live) { best[a] = bb; best_chi[a] = bchi; }
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
