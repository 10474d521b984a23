// tpc_tracklet.cuh -- a4 tracklet constructor (O4, steps 1-6; R9..R18, R23).
//
// One lane per start hit at a time.  The lane keeps the Kalman state and its bookkeeping in registers, the
// snapshot of the down pass in shared memory; rowhit[tracklet][row] lives in global memory (row fastest: a
// lane walks its own 32-byte sectors row by row, so L2 merges its writes).  Only rows first_row..last_row of
// a tracklet are ever read back, and every one of them is written here.
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

// Persistent warps; every lane owns one seed at a time and fetches the next one from a global counter as soon
// as its seed is finished ("lane refill"), so a warp stays full although seeds need between 1 and ~300 steps.
// The three passes of O4 (chain fit, up extrapolation, down pass) are folded into ONE step body
//     Propagate -> candidate (link | known hit | Search) -> Update -> bookkeeping
// driven by a per-lane phase, so that all lanes execute the expensive Kalman arithmetic together.  The order
// of floating-point operations of a seed is exactly the sequential algorithm's.
__global__ void __launch_bounds__(TC_THREADS) trackletConstructor(
    const uint32_t* __restrict__ off, DevParams P, RowTables T, const GridDesc* __restrict__ desc,
    const uint32_t* __restrict__ cell_start, const float2* __restrict__ syz, const uint32_t* __restrict__ s2o,
    const int32_t* __restrict__ cup, const uint32_t* __restrict__ start_pos, TrackletStore out, int64_t* __restrict__ cnt) {
  __shared__ float sx[MAX_ROWS];
  __shared__ int16_t sup[MAX_ROWS];
  __shared__ uint8_t sdead[MAX_ROWS];
  __shared__ float snap[22][TC_THREADS];     // state after the last Update of the down pass (O4 step 5)
  if (cnt[CNT_ERROR] != 0) return;
  const int R = P.n_rows;
  const int tid = threadIdx.x;
  for (int i = tid; i < R; i += blockDim.x) { sx[i] = T.row_x[i]; sup[i] = T.up_row[i]; sdead[i] = T.dead[i]; }
  __syncthreads();
  const int64_t nT = min(cnt[CNT_N_START], out.capT);
  const int64_t capT = out.capT;
  unsigned long long* work = (unsigned long long*)(cnt + CNT_WORK);

  KFState S;
  int phase = -1;                 // -1 wants a seed, -2 no seeds left, 0 chain fit, 1 up extrapolation, 2 down pass
  int64_t t = 0;
  int32_t* rowhit = nullptr;      // this tracklet's [n_rows] slice
  int r0 = 0, bsec = 0, rn = 0, rc = 0, lastw = 0, nhits = 0, miss = 0, snap_row = -1, rtop = 0;
  int32_t hlink = -1;

  for (;;) {
    if (phase == -1) {            // ---- fetch and initialise the next seed (O4 step 1) ----
      t = (int64_t)atomicAdd(work, 1ull);
      if (t >= nT) {
        phase = -2;
      } else {
        const uint32_t h0 = start_pos[t];
        const int b0 = bucketOf(off, P.n_buckets, h0);
        r0 = b0 % R;
        bsec = b0 - r0;
        rowhit = out.rowhit + t * R;
        hlink = cup[h0];
        rn = sup[r0];
        const float2 a = syz[h0], c = syz[hlink];
        S.x = sx[r0]; S.y = a.x; S.z = a.y;
        const float dx = sx[rn] - sx[r0], dy = c.x - a.x, dz = c.y - a.y;
        const float L = sqrtf(dx * dx + dy * dy);
        S.s = dy / L; S.t = dz / L; S.q = 0.0f;
        kfSetDiag(S, P.err2_y, P.err2_z, P);
        S.chi2 = 0.0f;
        rowhit[r0] = (int32_t)h0;
        nhits = 1; rc = r0; lastw = r0; miss = 0; snap_row = -1;
        out.sector[t] = bsec / R;
        phase = 0;
      }
    }
    __syncwarp();
    if (__all_sync(0xffffffffu, phase == -2)) break;

    // ---- one step: Propagate -> candidate -> Update ----
    const bool act = phase >= 0;
    const bool okp = act && kfPropagate(S, sx[act ? rn : 0], P);
    int32_t c = -1;
    bool known = false;
    if (okp) {
      if (phase == 0) { c = hlink; rc = rn; }
      else if (phase == 2 && rn >= r0) { c = rowhit[rn]; known = c != -1; }
    }
    const bool need_search = okp && c < 0;
    __syncwarp();
    if (need_search) c = kfSearch(S, desc[bsec + rn], cell_start, syz, s2o, P);
    __syncwarp();
    bool oku = false;
    if (okp && c >= 0) {
      const float2 m = syz[c];
      oku = kfUpdate(S, m.x, m.y, P);
    }
    __syncwarp();
    if (!act) continue;

    // ---- bookkeeping and phase transitions ----
    bool end_phase = !okp || (c >= 0 && !oku);       // Propagate or Update refused: the pass ends here
    bool turn = false;
    if (phase == 0) {
      if (oku) {
        for (int g = lastw + 1; g < rn; ++g) rowhit[g] = -1;
        rowhit[rn] = c;
        lastw = rn; ++nhits;
        hlink = cup[c];
        rn = sup[rn];
        if (hlink == -1) end_phase = true;
      }
      if (end_phase) {
        if (nhits < P.min_chain_hits) {
          out.status[t] = 0; out.nhits[t] = nhits; out.first_row[t] = -1; out.last_row[t] = -1;
          phase = -1;
        } else {
          phase = 1; miss = 0;
          rn = rc + 1;
          while (rn < R && sdead[rn]) ++rn;
          if (rn >= R) turn = true;
        }
      }
    } else if (phase == 1) {
      if (oku) {
        for (int g = lastw + 1; g < rn; ++g) rowhit[g] = -1;
        rowhit[rn] = c;
        lastw = rn; ++nhits; miss = 0;
      } else if (!end_phase) {
        if (++miss > P.max_row_gap) end_phase = true;
      }
      if (!end_phase) {
        ++rn;
        while (rn < R && sdead[rn]) ++rn;
        if (rn >= R) end_phase = true;
      }
      if (end_phase) turn = true;
    } else {
      if (!end_phase) {
        if (!known && (oku || rn < r0)) rowhit[rn] = oku ? c : -1;
        if (oku) {
          ++nhits; snap_row = rn;
          snap[0][tid] = S.x; snap[1][tid] = S.y; snap[2][tid] = S.z; snap[3][tid] = S.s; snap[4][tid] = S.t;
          snap[5][tid] = S.q; snap[6][tid] = S.chi2; snap[7][tid] = S.c00; snap[8][tid] = S.c10; snap[9][tid] = S.c11;
          snap[10][tid] = S.c20; snap[11][tid] = S.c21; snap[12][tid] = S.c22; snap[13][tid] = S.c30;
          snap[14][tid] = S.c31; snap[15][tid] = S.c32; snap[16][tid] = S.c33; snap[17][tid] = S.c40;
          snap[18][tid] = S.c41; snap[19][tid] = S.c42; snap[20][tid] = S.c43; snap[21][tid] = S.c44;
          if (rn < r0) miss = 0;
        } else if (rn < r0) {
          if (++miss > P.max_row_gap) end_phase = true;
        }
      }
      if (!end_phase) {
        --rn;
        while (rn >= 0 && sdead[rn]) { if (rn < r0) rowhit[rn] = -1; --rn; }
        if (rn < 0) end_phase = true;
      }
      if (end_phase) {            // O4 step 6: output = last snapshot
        if (snap_row < 0) {
          out.status[t] = 1; out.nhits[t] = 0; out.first_row[t] = -1; out.last_row[t] = -1;
        } else {
          out.status[t] = nhits >= P.min_tracklet_hits ? 2 : 1;
          out.nhits[t] = nhits; out.first_row[t] = snap_row; out.last_row[t] = rtop;
          out.x[t] = snap[0][tid]; out.chi2[t] = snap[6][tid];
#pragma unroll
          for (int i = 0; i < 5; ++i) out.par[i * capT + t] = snap[1 + i][tid];
#pragma unroll
          for (int i = 0; i < 15; ++i) out.cov[i * capT + t] = snap[7 + i][tid];
        }
        phase = -1;
      }
    }
    if (turn) {                   // O4 step 4: diffuse covariance, parameters kept (R17); down pass starts at rtop
      kfSetDiag(S, P.turn_var_scale * P.err2_y, P.turn_var_scale * P.err2_z, P);
      S.chi2 = 0.0f;
      rtop = lastw; rn = rtop;
      phase = 2; miss = 0; nhits = 0; snap_row = -1;
    }
  }
}

}  // namespace tpc
