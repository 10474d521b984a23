// tpc_refit.cuh -- a6: optional Kalman refit of the selected tracks over their kept clusters (DESIGN.md section 3 "O6",
// readings R28..R30; NEXT-2 of SURVEY.md 8(f); the paper names a track refit at PAPER.md L11 / L92).
//
// One thread per track.  up pass: state from the first two kept clusters as in O4 step 1, Propagate + Update through the
// others in ascending row -> outer state; turn (R17); down pass over all kept clusters -> inner state and chi2.
// Same Propagate / Update as the constructor (tpc_kalman.cuh), same order of operations as the formula sheet.
// The clusters are read from the caller's INPUT arrays by their global index (the track lists hold input indices);
// the row of a cluster follows from row_offset (R26): the lists are in ascending row, so the bucket only moves forward
// in the up pass and backward in the down pass.
#pragma once
#include "tpc_kalman.cuh"
#include "tpc_select.cuh"

namespace tpc {

struct RefitOut {
  int32_t* status;
  float *x_in, *par_in, *cov_in, *chi2, *x_out, *par_out, *cov_out;
};

__device__ __forceinline__ void refitStore(const KFState& S, int64_t k, int64_t cap, float* __restrict__ x,
                                           float* __restrict__ par, float* __restrict__ cov) {
  x[k] = S.x;
  par[0 * cap + k] = S.y; par[1 * cap + k] = S.z; par[2 * cap + k] = S.s; par[3 * cap + k] = S.t; par[4 * cap + k] = S.q;
  cov[0 * cap + k] = S.c00; cov[1 * cap + k] = S.c10; cov[2 * cap + k] = S.c11; cov[3 * cap + k] = S.c20;
  cov[4 * cap + k] = S.c21; cov[5 * cap + k] = S.c22; cov[6 * cap + k] = S.c30; cov[7 * cap + k] = S.c31;
  cov[8 * cap + k] = S.c32; cov[9 * cap + k] = S.c33; cov[10 * cap + k] = S.c40; cov[11 * cap + k] = S.c41;
  cov[12 * cap + k] = S.c42; cov[13 * cap + k] = S.c43; cov[14 * cap + k] = S.c44;
}

// Tracks are refitted in the order of their length (longest first) inside chunks of RF_CHUNK consecutive tracks, so that
// the 32 tracks of a warp need about the same number of steps AND the tracks in flight lie in a few sectors (the track
// order is the sector order): their cluster reads, random inside a sector, then stay in the L2.  Histogram of (chunk,
// length), exclusive scan (scanArrayInPlace), slots.  Order inside a bin is arbitrary.
constexpr int RF_BINS = 256;
#ifndef RF_CHUNK_
#define RF_CHUNK_ 32768
#endif
constexpr int RF_CHUNK = RF_CHUNK_;
__device__ __forceinline__ int64_t refitBin(int64_t k, uint32_t n) {
  return (k / RF_CHUNK) * RF_BINS + (RF_BINS - 1 - (int)min(n, (uint32_t)(RF_BINS - 1)));
}

__global__ void __launch_bounds__(256) refitCount(TrackOut o, uint32_t* __restrict__ hist, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= o.cap_tracks) return;
  atomicAdd(hist + refitBin(k, o.cl_offset[k + 1] - o.cl_offset[k]), 1u);
}

__global__ void __launch_bounds__(256) refitFill(TrackOut o, const uint32_t* __restrict__ start, uint32_t* __restrict__ fill,
                                                 uint32_t* __restrict__ order, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= cnt[CNT_N_TRACKS] || k >= o.cap_tracks) return;
  const int64_t b = refitBin(k, o.cl_offset[k + 1] - o.cl_offset[k]);
  order[start[b] + atomicAdd(fill + b, 1u)] = (uint32_t)k;
}

__global__ void __launch_bounds__(128) refitTracks(const uint32_t* __restrict__ off, const uint32_t* __restrict__ order, const float* __restrict__ y,
                                                   const float* __restrict__ z, DevParams P, RowTables T, TrackOut o,
                                                   RefitOut rf, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;               // truncated cluster lists cannot be refitted
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= cnt[CNT_N_TRACKS] || j >= o.cap_tracks) return;
  const int64_t k = order[j];
  const int64_t cap = o.cap_tracks;
  const uint32_t lo = o.cl_offset[k], hi = o.cl_offset[k + 1];
  const int n = (int)(hi - lo);
  KFState S{};
  bool ok = n >= 2;
  KFState So = S;
  if (ok) {
    const uint32_t* cl = o.cl_index + lo;
    const uint32_t c0 = cl[0], c1 = cl[1];
    int b = bucketOf(off, P.n_buckets, c0);
    const int bsec = b - b % P.n_rows;           // first bucket of the track's sector
    const float x0 = T.row_x[b - bsec];
    int b1 = b;
    while (__ldg(off + b1 + 1) <= c1) ++b1;
    {
      const float y0 = y[c0], z0 = z[c0];
      S.x = x0; S.y = y0; S.z = z0;
      const float dx = T.row_x[b1 - bsec] - x0, dy = y[c1] - y0, dz = z[c1] - z0;
      const float L = sqrtf(dx * dx + dy * dy);
      S.s = dy / L; S.t = dz / L; S.q = 0.0f;
    }
    kfSetDiag(S, P.err2_y, P.err2_z, P);
    S.chi2 = 0.0f;
    // Both passes are software-pipelined: the index and the coordinates of the NEXT cluster are requested before the
    // Kalman arithmetic of the current one (the input arrays are read at random: one DRAM latency per step otherwise).
    uint32_t cn = c1;
    float yn = y[c1], zn = z[c1];
    for (int i = 1; i < n && ok; ++i) {           // up pass
      const uint32_t c = cn;
      const float ym = yn, zm = zn;
      cn = cl[min(i + 1, n - 1)]; yn = y[cn]; zn = z[cn];      // unconditional: a conditional load would be waited for here
      while (__ldg(off + b + 1) <= c) ++b;
      ok = kfPropagate(S, T.row_x[b - bsec], P, [](float, float, float, float) {}) && kfUpdate(S, ym, zm, P);
    }
    So = S;
    if (ok) {                                     // turn (R17) and down pass
      kfSetDiag(S, P.turn_var_scale * P.err2_y, P.turn_var_scale * P.err2_z, P);
      S.chi2 = 0.0f;
      cn = cl[n - 1]; yn = y[cn]; zn = z[cn];
      for (int i = n - 1; i >= 0 && ok; --i) {
        const uint32_t c = cn;
        const float ym = yn, zm = zn;
        cn = cl[max(i - 1, 0)]; yn = y[cn]; zn = z[cn];
        while (__ldg(off + b) > c) --b;
        ok = kfPropagate(S, T.row_x[b - bsec], P, [](float, float, float, float) {}) && kfUpdate(S, ym, zm, P);
      }
    }
  }
  if (!ok) {                                      // R29: failed refit -> status 0, outputs zero
    S = KFState{}; So = KFState{};
  }
  rf.status[k] = ok ? 1 : 0;
  rf.chi2[k] = S.chi2;
  refitStore(S, k, cap, rf.x_in, rf.par_in, rf.cov_in);
  refitStore(So, k, cap, rf.x_out, rf.par_out, rf.cov_out);
}

}  // namespace tpc
