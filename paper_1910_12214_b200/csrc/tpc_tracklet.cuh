// tpc_tracklet.cuh -- a4 tracklet constructor (O4, steps 1-6; R9..R18, R23).
//
// One thread per start hit.  The thread keeps the Kalman state, the snapshot of the down pass and its
// bookkeeping in registers; rowhit[row][tracklet] lives in global memory (tracklet fastest, so threads of a
// warp that advance row by row together write coalesced).  Only rows first_row..last_row of a tracklet are
// ever read back, and every one of them is written here.
#pragma once
#include "tpc_kalman.cuh"
#include "tpc_links.cuh"

namespace tpc {

constexpr int TC_THREADS = 128;
constexpr int MAX_ROWS = 256;

// Search (O4): nearest cluster of the bucket inside the road around the predicted (y,z); key (d2, orig index).
__device__ __forceinline__ int32_t kfSearch(const KFState& S, const GridDesc& G, const uint32_t* __restrict__ cell_start,
                                            const float2* __restrict__ syz, const uint32_t* __restrict__ s2o,
                                            const DevParams& P) {
  float ry = P.road_sigma * sqrtf(S.c00 + P.err2_y);
  float rz = P.road_sigma * sqrtf(S.c11 + P.err2_z);
  if (!(ry >= P.road_min)) ry = P.road_min;
  if (ry > P.road_max) ry = P.road_max;
  if (!(rz >= P.road_min)) rz = P.road_min;
  if (rz > P.road_max) rz = P.road_max;
  int32_t best = -1;
  float bestd = 0.0f;
  const float yp = S.y, zp = S.z;
  forWindow(G, cell_start, syz, yp, zp, ry, rz, [&](uint32_t c, float yc, float zc) {
    const float dy = yc - yp, dz = zc - zp;
    const float d2 = dy * dy + dz * dz;
    if (best < 0 || d2 < bestd || (d2 == bestd && __ldg(s2o + c) < __ldg(s2o + best))) { best = (int32_t)c; bestd = d2; }
  });
  return best;
}

__global__ void __launch_bounds__(TC_THREADS) trackletConstructor(
    const uint32_t* __restrict__ off, DevParams P, RowTables T, const GridDesc* __restrict__ desc,
    const uint32_t* __restrict__ cell_start, const float2* __restrict__ syz, const uint32_t* __restrict__ s2o,
    const int32_t* __restrict__ cup, const uint32_t* __restrict__ start_pos, TrackletStore out,
    const int64_t* __restrict__ cnt) {
  __shared__ float sx[MAX_ROWS];
  __shared__ int16_t sup[MAX_ROWS];
  __shared__ uint8_t sdead[MAX_ROWS];
  if (cnt[CNT_ERROR] != 0) return;
  const int R = P.n_rows;
  for (int i = threadIdx.x; i < R; i += blockDim.x) { sx[i] = T.row_x[i]; sup[i] = T.up_row[i]; sdead[i] = T.dead[i]; }
  __syncthreads();
  const int64_t nT = min(cnt[CNT_N_START], out.capT);
  const int64_t capT = out.capT;
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nT; t += (int64_t)gridDim.x * blockDim.x) {
    const uint32_t h0 = start_pos[t];
    const int b0 = bucketOf(off, P.n_buckets, h0);
    const int r0 = b0 % R;
    const int bsec = b0 - r0;                 // bucket of row 0 of this sector
    int32_t* rowhit = out.rowhit + t;         // row stride capT
    KFState S;
    // 1. initialise from the first link
    const int32_t h1 = cup[h0];
    int r = sup[r0];
    {
      const float2 a = syz[h0], c = syz[h1];
      S.x = sx[r0]; S.y = a.x; S.z = a.y;
      const float dx = sx[r] - sx[r0], dy = c.x - a.x, dz = c.y - a.y;
      const float L = sqrtf(dx * dx + dy * dy);
      S.s = dy / L; S.t = dz / L; S.q = 0.0f;
    }
    kfSetDiag(S, P.err2_y, P.err2_z, P);
    S.chi2 = 0.0f;
    rowhit[(int64_t)r0 * capT] = (int32_t)h0;
    int nhits = 1, rc = r0, lastw = r0;
    // 2. fit along the link chain
    for (int32_t h = h1; h != -1;) {
      if (!kfPropagate(S, sx[r], P)) break;
      rc = r;
      const float2 c = syz[h];
      if (!kfUpdate(S, c.x, c.y, P)) break;
      for (int g = lastw + 1; g < r; ++g) rowhit[(int64_t)g * capT] = -1;
      rowhit[(int64_t)r * capT] = h;
      lastw = r; ++nhits;
      h = cup[h];
      r = sup[r];
    }
    out.sector[t] = bsec / R;
    if (nhits < P.min_chain_hits) {
      out.status[t] = 0; out.nhits[t] = nhits; out.first_row[t] = -1; out.last_row[t] = -1;
      continue;
    }
    // 3. extrapolate upwards, picking up clusters through the grid
    int miss = 0;
    for (r = rc + 1; r < R; ++r) {
      if (sdead[r]) continue;
      if (!kfPropagate(S, sx[r], P)) break;
      const int32_t c = kfSearch(S, desc[bsec + r], cell_start, syz, s2o, P);
      if (c >= 0) {
        const float2 m = syz[c];
        if (!kfUpdate(S, m.x, m.y, P)) break;
        for (int g = lastw + 1; g < r; ++g) rowhit[(int64_t)g * capT] = -1;
        rowhit[(int64_t)r * capT] = c;
        lastw = r; ++nhits; miss = 0;
      } else if (++miss > P.max_row_gap) break;
    }
    // 4. turn: diffuse covariance, parameters kept as the linearisation point (R17)
    kfSetDiag(S, P.turn_var_scale * P.err2_y, P.turn_var_scale * P.err2_z, P);
    S.chi2 = 0.0f;
    const int rtop = lastw;
    // 5. down pass over all collected hits, filling gaps and extending below the start row
    KFState snap = S;
    int snap_row = -1, nh = 0;
    miss = 0;
    for (r = rtop; r >= 0; --r) {
      if (sdead[r]) { if (r < r0) rowhit[(int64_t)r * capT] = -1; continue; }
      if (!kfPropagate(S, sx[r], P)) break;
      int32_t c = (r >= r0) ? rowhit[(int64_t)r * capT] : -1;
      const bool known = c != -1;
      if (!known) c = kfSearch(S, desc[bsec + r], cell_start, syz, s2o, P);
      bool ok = false;
      if (c >= 0) {
        const float2 m = syz[c];
        if (!kfUpdate(S, m.x, m.y, P)) break;
        ok = true;
      }
      if (!known && (ok || r < r0)) rowhit[(int64_t)r * capT] = ok ? c : -1;
      if (ok) {
        ++nh; snap = S; snap_row = r;
        if (r < r0) miss = 0;
      } else if (r < r0) {
        if (++miss > P.max_row_gap) break;
      }
    }
    // 6. output = last snapshot (state at the innermost attached row)
    if (snap_row < 0) {
      out.status[t] = 1; out.nhits[t] = 0; out.first_row[t] = -1; out.last_row[t] = -1;
      continue;
    }
    out.status[t] = nh >= P.min_tracklet_hits ? 2 : 1;
    out.nhits[t] = nh; out.first_row[t] = snap_row; out.last_row[t] = rtop;
    out.x[t] = snap.x; out.chi2[t] = snap.chi2;
    out.par[0 * capT + t] = snap.y; out.par[1 * capT + t] = snap.z; out.par[2 * capT + t] = snap.s;
    out.par[3 * capT + t] = snap.t; out.par[4 * capT + t] = snap.q;
    float* cv = out.cov + t;
    cv[0 * capT] = snap.c00; cv[1 * capT] = snap.c10; cv[2 * capT] = snap.c11; cv[3 * capT] = snap.c20;
    cv[4 * capT] = snap.c21; cv[5 * capT] = snap.c22; cv[6 * capT] = snap.c30; cv[7 * capT] = snap.c31;
    cv[8 * capT] = snap.c32; cv[9 * capT] = snap.c33; cv[10 * capT] = snap.c40; cv[11 * capT] = snap.c41;
    cv[12 * capT] = snap.c42; cv[13 * capT] = snap.c43; cv[14 * capT] = snap.c44;
  }
}

}  // namespace tpc
