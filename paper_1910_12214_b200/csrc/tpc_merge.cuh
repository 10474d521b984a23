// tpc_merge.cuh -- a7: optional links between track segments (DESIGN.md section 3 "O7", readings R31..R33; NEXT-1 of
// SURVEY.md 8(f); PAPER.md L92 stresses the merging and gives no method).
//
// A refitted track a (outer state) may continue in a refitted track b (inner state) of the same sector further out, or
// of the azimuthal neighbour sector.  chi2(a, b) = diagonal chi2 of a's outer state -- rotated into b's frame if
// needed, propagated to b's reference plane -- against b's inner state.  next(a) = admissible b of minimal (chi2, id),
// prev(b) = admissible a of minimal (chi2, id); a link is kept when both agree.
//
// Organisation: the tracks are bucketed by (sector, first kept row, bin of the dip t of their inner state).  The dip and
// curvature terms of the chi2 need no transport -- Rotate and Propagate leave t, q, C33 and C44 as they are -- so they are
// tested first, on 16-byte records packed in list order, and only the dip bins that can hold a b whose dip term alone
// stays below the cut are visited: the terms are non-negative and rounding is monotone, so the sum could only be larger,
// and the window uses the largest dip variance of the (sector, row) (plus rounding slack; badly measured dips sit in one
// extra bin that is always visited), so it is a superset of every admissible b -- no result changes (same argument as
// R3).  All b of a (sector, row) share their reference plane: a is propagated once per ROW that has a surviving candidate,
// which is a handful of the 132 rows in reach.  prev(b) is an atomicMin over (chi2 bits, a).
#pragma once
#include "tpc_kalman.cuh"
#include "tpc_refit.cuh"

namespace tpc {

struct MergeIn {            // refit outputs and track bookkeeping (device, SoA with stride cap)
  int64_t cap;
  const int32_t *status, *sector, *first_row, *last_row;
  const float *x_in, *par_in, *cov_in, *x_out, *par_out, *cov_out;
};
struct MergeOut {
  int32_t *next, *prev, *head;
  float* chi2;
};
constexpr int MG_NTB = 64;                   // dip bins over [-MG_TMAX, MG_TMAX] (clamped outside)
constexpr float MG_TMAX = 2.0f;
constexpr float MG_VWIDE = 2e-5f;            // inner states with a larger dip variance go to one extra bin, always visited
constexpr int MG_BINS = MG_NTB + 1;

__device__ __forceinline__ int mergeDipBin(float t) { return cellCoord(t, -MG_TMAX, (float)MG_NTB / (2.0f * MG_TMAX), MG_NTB); }
__device__ __forceinline__ int mergeBucket(int sr, float t, float var_t) {
  return sr * MG_BINS + (var_t <= MG_VWIDE ? mergeDipBin(t) : MG_NTB);
}

struct MergeParams {
  int32_t max_row_gap, back_rows;
  float chi2_max, ca, sa;    // ca, sa = (float)cos / sin of 20 degrees
};

// per track: clear the outputs, count the refitted tracks per (sector, first row)
__global__ void __launch_bounds__(256) mergeCount(MergeIn in, MergeOut out, DevParams P, RowTables T,
                                                  uint32_t* __restrict__ bucket_cnt, uint32_t* __restrict__ order_cnt,
                                                  uint32_t* __restrict__ max_var, int32_t* __restrict__ best_b, unsigned long long* __restrict__ key_a,
                                                  const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap) return;
  out.next[k] = -1; out.prev[k] = -1; out.head[k] = (int32_t)k; out.chi2[k] = 0.0f;
  best_b[k] = -1; key_a[k] = ~0ull;
  if (in.status[k] == 1) {
    const int sr = in.sector[k] * P.n_rows + in.first_row[k];
    const float vt = in.cov_in[9 * in.cap + k];
    atomicAdd(bucket_cnt + mergeBucket(sr, in.par_in[3 * in.cap + k], vt), 1u);
    // largest binned dip variance of the (sector, row): positive floats order like their bit patterns
    if (vt <= MG_VWIDE) atomicMax(max_var + sr, __float_as_uint(vt));
    // the order in which mergeMatch takes the tracks a: by (sector, last row, dip bin) of the OUTER state
    atomicAdd(order_cnt + mergeBucket(in.sector[k] * P.n_rows + in.last_row[k], in.par_out[3 * in.cap + k], in.cov_out[9 * in.cap + k]), 1u);
  }
}

// per track: its slot in the bucket list (order inside a bucket is arbitrary: every argmin below breaks ties by id)
__global__ void __launch_bounds__(256) mergeFill(MergeIn in, DevParams P, RowTables T, const uint32_t* __restrict__ bucket_start,
                                                 uint32_t* __restrict__ bucket_fill, uint32_t* __restrict__ list,
                                                 float4* __restrict__ rec, const uint32_t* __restrict__ order_start,
                                                 uint32_t* __restrict__ order_fill, uint32_t* __restrict__ order,
                                                 const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap || in.status[k] != 1) return;
  {
    const int o = mergeBucket(in.sector[k] * P.n_rows + in.last_row[k], in.par_out[3 * in.cap + k], in.cov_out[9 * in.cap + k]);
    order[order_start[o] + atomicAdd(order_fill + o, 1u)] = (uint32_t)k;
  }
  const float t = in.par_in[3 * in.cap + k], vt = in.cov_in[9 * in.cap + k];
  const int b = mergeBucket(in.sector[k] * P.n_rows + in.first_row[k], t, vt);
  const uint32_t slot = bucket_start[b] + atomicAdd(bucket_fill + b, 1u);
  list[slot] = (uint32_t)k;
  rec[slot] = make_float4(t, in.par_in[4 * in.cap + k], vt, in.cov_in[14 * in.cap + k]);   // what the first tests read
}

// O7 Rotate(alpha) with (ca, sa); returns false (state untouched) if |sin phi'| would reach max_sinphi
__device__ __forceinline__ bool kfRotate(KFState& S, float ca, float sa, const DevParams& P) {
  const float s = S.s, t = S.t;
  const float c = sqrtf(1.0f - s * s);
  const float s1 = s * ca - c * sa;
  if (!(fabsf(s1) < P.max_sinphi)) return false;
  const float c1 = sqrtf(1.0f - s1 * s1);
  const float x1 = S.x * ca + S.y * sa;
  const float y1 = S.y * ca - S.x * sa;
  const float jy = c / c1, jz = -(sa * t) / c1, js = c1 / c, jq = -((S.q * P.b) * sa);
  const float C00 = S.c00, C10 = S.c10, C11 = S.c11, C20 = S.c20, C21 = S.c21, C22 = S.c22, C30 = S.c30, C31 = S.c31,
              C32 = S.c32, C40 = S.c40, C41 = S.c41, C42 = S.c42;
  const float m2 = jq * C00 + js * C20;
  S.c00 = (jy * jy) * C00;
  S.c10 = jy * (jz * C00 + C10);
  S.c11 = ((jz * jz) * C00 + (2.0f * jz) * C10) + C11;
  S.c20 = jy * m2;
  S.c21 = jz * m2 + (jq * C10 + js * C21);
  S.c22 = ((jq * jq) * C00 + ((2.0f * jq) * js) * C20) + (js * js) * C22;
  S.c30 = jy * C30;
  S.c31 = jz * C30 + C31;
  S.c32 = jq * C30 + js * C32;
  S.c40 = jy * C40;
  S.c41 = jz * C40 + C41;
  S.c42 = jq * C40 + js * C42;
  S.x = x1; S.y = y1; S.s = s1;
  return true;
}

__device__ __forceinline__ KFState mergeLoad(int64_t k, int64_t cap, const float* __restrict__ x,
                                             const float* __restrict__ par, const float* __restrict__ cov) {
  KFState S{};
  S.x = x[k];
  S.y = par[0 * cap + k]; S.z = par[1 * cap + k]; S.s = par[2 * cap + k]; S.t = par[3 * cap + k]; S.q = par[4 * cap + k];
  S.c00 = cov[0 * cap + k]; S.c10 = cov[1 * cap + k]; S.c11 = cov[2 * cap + k]; S.c20 = cov[3 * cap + k];
  S.c21 = cov[4 * cap + k]; S.c22 = cov[5 * cap + k]; S.c30 = cov[6 * cap + k]; S.c31 = cov[7 * cap + k];
  S.c32 = cov[8 * cap + k]; S.c33 = cov[9 * cap + k]; S.c40 = cov[10 * cap + k]; S.c41 = cov[11 * cap + k];
  S.c42 = cov[12 * cap + k]; S.c43 = cov[13 * cap + k]; S.c44 = cov[14 * cap + k];
  return S;
}

__device__ __forceinline__ int64_t live_guard(int64_t a, int64_t cap) { return a < cap ? a : 0; }

// one thread per track a: best continuation b of a, and a's bid for every admissible b
__global__ void __launch_bounds__(128) mergeMatch(MergeIn in, DevParams P, RowTables T, MergeParams M,
                                                  const uint32_t* __restrict__ bucket_start,
                                                  const uint32_t* __restrict__ max_var,
                                                  const uint32_t* __restrict__ list, const float4* __restrict__ rec,
                                                  const uint32_t* __restrict__ order_start, const uint32_t* __restrict__ order,
                                                  int32_t* __restrict__ best_b, float* __restrict__ chi_b,
                                                  unsigned long long* __restrict__ key_a, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  // the tracks a are taken by (sector, last row, dip bin) of their outer state: the lanes of a warp walk nearly the
  // same rows and the same runs of candidates
  // Lanes without a track stay in the loops (predicated off): the row loop has the same trip count for every lane and
  // reconverges at __syncwarp(), so the lanes set up a row together however many candidates each had on the last one.
  const int64_t slot = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = slot < order_start[(int64_t)P.n_buckets * MG_BINS];
  const int64_t a = live ? order[slot] : 0;
  const int64_t cap = in.cap;
  const int R = P.n_rows;
  const int sa_sec = live ? in.sector[a] : 0, la = live ? in.last_row[a] : 0;
  KFState A0{};
  if (live) A0 = mergeLoad(a, cap, in.x_out, in.par_out, in.cov_out);
  int32_t bb = -1;
  float bchi = 0.0f;
  const int n_it = M.back_rows + M.max_row_gap + 1;      // rows la - back_rows .. la + max_row_gap
  for (int rel = 0; rel <= 2; ++rel) {           // 0 same sector, 1 next sector (+20 degrees), 2 previous sector
    if (rel != 0 && P.n_sectors != 36) break;    // uniform
    int sb = sa_sec;
    KFState Ar = A0;
    bool rel_ok = live;
    if (rel != 0) {
      const int side = sa_sec / 18, j = sa_sec - side * 18;
      sb = side * 18 + (rel == 1 ? (j + 1) % 18 : (j + 17) % 18);
      rel_ok = live && kfRotate(Ar, M.ca, rel == 1 ? M.sa : -M.sa, P);
    }
    const int r_lo = max(0, la + (rel == 0 ? 1 : -M.back_rows)), r_hi = min(R - 1, la + M.max_row_gap);
    for (int it = 0; it < n_it; ++it) {
      __syncwarp();
      const int r = la - M.back_rows + it;
      if (!(rel_ok && r >= r_lo && r <= r_hi)) continue;
      const int sr = sb * R + r;
      const uint32_t* bs = bucket_start + sr * MG_BINS;
      // dip bins that can hold an admissible b: |t_a - t_b| <= sqrt(chi2_max * (C33_a + max C33_b)), with slack; a window
      // that is not >= 0 means no positive denominator is possible among the binned b
      const float w = sqrtf(M.chi2_max * (Ar.c33 + __uint_as_float(max_var[sr]))) * 1.0001f + 1e-6f;
      const bool any = w >= 0.0f;
      const uint32_t j0 = bs[MG_NTB], j1 = bs[MG_BINS];        // the b with a wide dip variance: always visited
      const uint32_t i0 = any ? bs[mergeDipBin(Ar.t - w)] : j0, i1 = any ? bs[mergeDipBin(Ar.t + w) + 1] : j0;
      KFState S = Ar;
      int state = 0;                               // 0 not propagated to this row yet, 1 done, 2 refused
      for (uint32_t ii = i0; ii < i1 + (j1 - j0) && state != 2; ++ii) {
        const uint32_t i = ii < i1 ? ii : j0 + (ii - i1);
        // The dip and curvature terms need no transport (see the header); one of them above the cut decides.
        const float4 rc = __ldg(rec + i);          // t, q, C33, C44 of the candidate
        const float den3 = Ar.c33 + rc.z, den4 = Ar.c44 + rc.w;
        const float d3 = Ar.t - rc.x, d4 = Ar.q - rc.y;
        const float t3 = (d3 * d3) / den3, t4 = (d4 * d4) / den4;
        if (t3 > M.chi2_max || t4 > M.chi2_max) continue;
        const int64_t b = list[i];
        if (b == a) continue;
        if (state == 0) state = kfPropagate(S, T.row_x[r], P, [](float, float, float, float) {}) ? 1 : 2;
        if (state == 2) break;
        // the five terms in the order of Match: y, z, s, t, q
        const float pa[3] = {S.y, S.z, S.s};
        const float ca[3] = {S.c00, S.c11, S.c22};
        const int ci[3] = {0, 2, 5};
        bool ok = true;
        float sum = 0.0f;
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          const float den = ca[q] + in.cov_in[ci[q] * cap + b];
          if (!(den > 0.0f)) { ok = false; break; }
          const float d = pa[q] - in.par_in[q * cap + b];
          sum = sum + (d * d) / den;
          if (!(sum <= M.chi2_max)) { ok = false; break; }       // the terms are non-negative: it can only grow
        }
        if (!ok || !(den3 > 0.0f) || !(den4 > 0.0f)) continue;
        sum = sum + t3;
        sum = sum + t4;
        if (!(sum <= M.chi2_max)) continue;
        if (bb < 0 || sum < bchi || (sum == bchi && (int32_t)b < bb)) { bb = (int32_t)b; bchi = sum; }
        atomicMin(key_a + b, ((unsigned long long)__float_as_uint(sum) << 32) | (unsigned long long)(uint32_t)a);
      }
    }
  }
  if (live) { best_b[a] = bb; chi_b[a] = bchi; }
}

// a link is kept when next(a) = b and prev(b) = a (R33)
__global__ void __launch_bounds__(256) mergeLink(MergeIn in, MergeOut out, const int32_t* __restrict__ best_b,
                                                 const float* __restrict__ chi_b,
                                                 const unsigned long long* __restrict__ key_a,
                                                 const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= cnt[CNT_N_TRACKS] || a >= in.cap) return;
  const int32_t b = best_b[a];
  if (b >= 0 && (uint32_t)(key_a[b] & 0xffffffffull) == (uint32_t)a) {
    out.next[a] = b; out.prev[b] = (int32_t)a; out.chi2[a] = chi_b[a];
  }
}

// head(k) = first track of k's chain (chains are a handful of segments long)
__global__ void __launch_bounds__(256) mergeHead(MergeIn in, MergeOut out, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t nt = min(cnt[CNT_N_TRACKS], in.cap);
  if (k >= nt) return;
  int64_t h = k;
  for (int64_t guard = 0; guard < nt; ++guard) {
    const int32_t p = out.prev[h];
    if (p < 0) break;
    h = p;
  }
  out.head[k] = (int32_t)h;
}

}  // namespace tpc
