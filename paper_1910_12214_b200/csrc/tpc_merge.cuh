// tpc_merge.cuh -- a7: optional links between track segments (DESIGN.md section 3 "O7", readings R31..R33; NEXT-1 of
// SURVEY.md 8(f); PAPER.md L92 stresses the merging and gives no method).
//
// A refitted track a (outer state) may continue in a refitted track b (inner state) of the same sector further out, or
// of the azimuthal neighbour sector.  chi2(a, b) = diagonal chi2 of a's outer state -- rotated into b's frame if
// needed, propagated to b's reference plane -- against b's inner state.  next(a) = admissible b of minimal (chi2, id),
// prev(b) = admissible a of minimal (chi2, id); a link is kept when both agree.
//
// Organisation: the tracks are bucketed by (sector, first kept row, z bin, y bin of their inner state) -- all b of a
// (sector, row) share their reference plane, so a is propagated once per candidate ROW, not once per pair, and only the
// bins that can hold a b whose y or z term alone stays below the cut are visited: the terms are non-negative, so the
// sum could only be larger, and the window uses the largest inner variances of the row (plus rounding slack), so it is a
// superset of every admissible b -- no result changes (same argument as R3).  prev(b) is an atomicMin over (chi2 bits, a).
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
constexpr int MG_NYB = 32, MG_NZB = 16;     // y / z bins of the inner states per (sector, row)
constexpr int MG_GROUP = 1;                  // lanes per track in mergeMatch (more lanes only repeat the 132 Propagates: 4 -> 14.2 ms against 13.2)

__device__ __forceinline__ int mergeBucket(int sr, float y, float z, float x_row, const DevParams& P) {
  const float hw = x_row * P.tan_half_sector;
  const int by = cellCoord(y, -hw, (float)MG_NYB / (2.0f * hw), MG_NYB);
  const int bz = cellCoord(z, P.z_min, (float)MG_NZB / (P.z_max - P.z_min), MG_NZB);
  return (sr * MG_NZB + bz) * MG_NYB + by;
}

struct MergeParams {
  int32_t max_row_gap, back_rows;
  float chi2_max, ca, sa;    // ca, sa = (float)cos / sin of 20 degrees
};

// per track: clear the outputs, count the refitted tracks per (sector, first row)
__global__ void __launch_bounds__(256) mergeCount(MergeIn in, MergeOut out, DevParams P, RowTables T,
                                                  uint32_t* __restrict__ bucket_cnt, uint32_t* __restrict__ max_var,
                                                  int32_t* __restrict__ best_b, unsigned long long* __restrict__ key_a,
                                                  const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap) return;
  out.next[k] = -1; out.prev[k] = -1; out.head[k] = (int32_t)k; out.chi2[k] = 0.0f;
  best_b[k] = -1; key_a[k] = ~0ull;
  if (in.status[k] == 1) {
    const int r = in.first_row[k], sr = in.sector[k] * P.n_rows + r;
    atomicAdd(bucket_cnt + mergeBucket(sr, in.par_in[k], in.par_in[in.cap + k], T.row_x[r], P), 1u);
    // largest inner variances of the (sector, row): positive floats order like their bit patterns
    atomicMax(max_var + 2 * sr, __float_as_uint(in.cov_in[k]));
    atomicMax(max_var + 2 * sr + 1, __float_as_uint(in.cov_in[2 * in.cap + k]));
  }
}

// per track: its slot in the bucket list (order inside a bucket is arbitrary: every argmin below breaks ties by id)
__global__ void __launch_bounds__(256) mergeFill(MergeIn in, DevParams P, RowTables T, const uint32_t* __restrict__ bucket_start,
                                                 uint32_t* __restrict__ bucket_fill, uint32_t* __restrict__ list,
                                                 const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap || in.status[k] != 1) return;
  const int r = in.first_row[k];
  const int b = mergeBucket(in.sector[k] * P.n_rows + r, in.par_in[k], in.par_in[in.cap + k], T.row_x[r], P);
  list[bucket_start[b] + atomicAdd(bucket_fill + b, 1u)] = (uint32_t)k;
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
                                                  const uint32_t* __restrict__ list, int32_t* __restrict__ best_b,
                                                  float* __restrict__ chi_b, unsigned long long* __restrict__ key_a,
                                                  const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  // MG_GROUP lanes per track: they carry the same state (the Propagate of a row is redundant but uniform) and share the
  // candidates of the bins; their best continuations are merged by shuffles at the end.
  const int64_t a = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / MG_GROUP;
  const int sub = threadIdx.x % MG_GROUP;
  // Lanes without a track stay in the loops (predicated off): the row loop below has the same trip count for every
  // lane and reconverges at __syncwarp(), so the 32 lanes run the Propagate of a row together.
  const bool live = a < cnt[CNT_N_TRACKS] && a < in.cap && in.status[live_guard(a, in.cap)] == 1;
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
      bool act = rel_ok && r >= r_lo && r <= r_hi;
      const int sr = act ? sb * R + r : 0;
      const float vy = act ? __uint_as_float(max_var[2 * sr]) : 0.0f;
      act = act && vy != 0.0f;                     // no refitted track starts on this (sector, row)
      KFState S = Ar;
      const float xr = T.row_x[act ? r : 0];
      const bool okp = kfPropagate(S, act ? xr : S.x, P, [](float, float, float, float) {});
      if (!(act && okp)) continue;
      // bins that can hold an admissible b: |dy| <= sqrt(chi2_max * (C00 + max C00_b)), likewise z (with slack)
      const float wy = sqrtf(M.chi2_max * (S.c00 + vy)) * 1.0001f + 1e-6f;
      const float wz = sqrtf(M.chi2_max * (S.c11 + __uint_as_float(max_var[2 * sr + 1]))) * 1.0001f + 1e-6f;
      if (!(wy >= 0.0f) || !(wz >= 0.0f)) continue;      // a non-positive variance of a: every denominator test fails below anyway
      const float hw = xr * P.tan_half_sector;
      const float iby = (float)MG_NYB / (2.0f * hw), ibz = (float)MG_NZB / (P.z_max - P.z_min);
      const int by0 = cellCoord(S.y - wy, -hw, iby, MG_NYB), by1 = cellCoord(S.y + wy, -hw, iby, MG_NYB);
      const int bz0 = cellCoord(S.z - wz, P.z_min, ibz, MG_NZB), bz1 = cellCoord(S.z + wz, P.z_min, ibz, MG_NZB);
      for (int bz = bz0; bz <= bz1; ++bz) {
      const uint32_t* row = bucket_start + (sr * MG_NZB + bz) * MG_NYB;
      const uint32_t k0 = row[by0], k1 = row[by1 + 1];
      for (uint32_t i = k0 + sub; i < k1; i += MG_GROUP) {
        const int64_t b = list[i];
        if (b == a) continue;
        // the y term first: it alone decides for almost every pair of the bucket
        const float den0 = S.c00 + in.cov_in[0 * cap + b];
        if (!(den0 > 0.0f)) continue;
        const float d0 = S.y - in.par_in[0 * cap + b];
        float sum = 0.0f + (d0 * d0) / den0;
        if (!(sum <= M.chi2_max)) continue;
        const float pa[4] = {S.z, S.s, S.t, S.q};
        const float ca[4] = {S.c11, S.c22, S.c33, S.c44};
        const int ci[4] = {2, 5, 9, 14};
        bool ok = true;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const float den = ca[q] + in.cov_in[ci[q] * cap + b];
          if (!(den > 0.0f)) { ok = false; break; }
          const float d = pa[q] - in.par_in[(q + 1) * cap + b];
          sum = sum + (d * d) / den;
        }
        if (!ok || !(sum <= M.chi2_max)) continue;
        if (bb < 0 || sum < bchi || (sum == bchi && (int32_t)b < bb)) { bb = (int32_t)b; bchi = sum; }
        atomicMin(key_a + b, ((unsigned long long)__float_as_uint(sum) << 32) | (unsigned long long)(uint32_t)a);
      }
      }
    }
  }
  __syncwarp();
#pragma unroll
  for (int d = 1; d < MG_GROUP; d <<= 1) {         // minimal (chi2, id) over the lanes of the group
    const int32_t ob = __shfl_xor_sync(0xffffffffu, bb, d);
    const float oc = __shfl_xor_sync(0xffffffffu, bchi, d);
    if (ob >= 0 && (bb < 0 || oc < bchi || (oc == bchi && ob < bb))) { bb = ob; bchi = oc; }
  }
  if (live && sub == 0) { best_b[a] = bb; chi_b[a] = bchi; }
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
