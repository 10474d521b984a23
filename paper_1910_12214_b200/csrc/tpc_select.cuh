// tpc_select.cuh -- a5 tracklet selector (O5; R19..R22, R27) and the optional per-stage exports.
//
// owner(c) = accepted tracklet of highest priority containing c; priority: more hits, then smaller chi2
// (fp32 compare), then smaller tracklet id.  Implemented as atomicMax over a key whose integer order is
// that priority: chi2 >= 0, so its IEEE bit pattern orders like its value.
//   packed key (n_rows <= 255, ids < 2^24):  nhits[63:56] | ~chi2bits[55:24] | ~id[23:0]
//   wide keys  (any id):  pass 1 atomicMax(nhits[63:32] | ~chi2bits[31:0]); pass 2 atomicMin(id) among equals.
#pragma once
#include "tpc_common.cuh"

namespace tpc {

__device__ __forceinline__ unsigned long long selKey(int nhits, float chi2, uint32_t id, bool wide) {
  const unsigned long long inv = (unsigned long long)(~__float_as_uint(chi2));
  if (wide) return ((unsigned long long)(uint32_t)nhits << 32) | inv;
  return ((unsigned long long)(uint32_t)nhits << 56) | (inv << 24) | (unsigned long long)((~id) & 0xFFFFFFu);
}

// four consecutive row hits of a tracklet's slice starting at row rb (a multiple of 4): one 16-byte load when the slices
// are 16-byte aligned (n_rows a multiple of 4), rows outside [f, r1] masked to -1
__device__ __forceinline__ void rowHits4(const int32_t* __restrict__ row, int n_rows, int rb, int f, int r1, int32_t c4[4]) {
  if ((n_rows & 3) == 0) {
    const int4 v = *reinterpret_cast<const int4*>(row + rb);
    c4[0] = v.x; c4[1] = v.y; c4[2] = v.z; c4[3] = v.w;
  } else {
#pragma unroll
    for (int k = 0; k < 4; ++k) c4[k] = rb + k < n_rows ? row[rb + k] : -1;
  }
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (rb + k < f || rb + k > r1) c4[k] = -1;
}

__global__ void __launch_bounds__(128) selectClaim(TrackletStore tl, unsigned long long* __restrict__ owner_key,
                                                   int wide, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nT = min(cnt[CNT_N_START], tl.capT);
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nT || tl.status[t] != 2) return;
  const unsigned long long key = selKey(tl.nhits[t], tl.chi2[t], (uint32_t)t, wide != 0);
  const int f = tl.first_row[t], r1 = tl.last_row[t];
  const int32_t* row = tl.rowhit + t * tl.n_rows;
  for (int rb = f & ~3; rb <= r1; rb += 4) {
    int32_t c4[4];
    rowHits4(row, tl.n_rows, rb, f, r1, c4);
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (c4[k] >= 0) atomicMax(owner_key + c4[k], key);
  }
}

// wide keys only: among the tracklets whose (nhits, chi2) equal the winning pair, the smallest id owns.
__global__ void __launch_bounds__(128) selectClaimId(TrackletStore tl, const unsigned long long* __restrict__ owner_key,
                                                     uint32_t* __restrict__ owner_id, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nT = min(cnt[CNT_N_START], tl.capT);
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nT || tl.status[t] != 2) return;
  const unsigned long long key = selKey(tl.nhits[t], tl.chi2[t], (uint32_t)t, true);
  const int r1 = tl.last_row[t];
  for (int r = tl.first_row[t]; r <= r1; ++r) {
    const int32_t c = tl.rowhit[t * tl.n_rows + r];
    if (c >= 0 && owner_key[c] == key) atomicMin(owner_id + c, (uint32_t)t);
  }
}

__device__ __forceinline__ bool owns(int32_t c, unsigned long long key, uint32_t t, int wide,
                                     const unsigned long long* __restrict__ owner_key,
                                     const uint32_t* __restrict__ owner_id) {
  if (owner_key[c] != key) return false;
  return !wide || owner_id[c] == t;
}

// per tracklet: kept = hits it owns; a track iff kept >= min_track_hits (single pass, R21).
// tsel[t] = is_track | kept << 32 (0 when not a track).  Also counts accepted tracklets and their hits.
// NOTE: rewrites the front of every accepted tracklet's row-hit slice (exports of the row hits run before this kernel).
__global__ void __launch_bounds__(128) selectCount(TrackletStore tl, const unsigned long long* __restrict__ owner_key,
                                                   const uint32_t* __restrict__ owner_id, int wide, int min_track_hits,
                                                   unsigned long long* __restrict__ tsel, int32_t* __restrict__ kept_first,
                                                   int32_t* __restrict__ kept_last, int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nT = min(cnt[CNT_N_START], tl.capT);
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long acc = 0;   // accepted | hits << 32
  if (t < nT) {
    unsigned long long sel = 0;
    if (tl.status[t] == 2) {
      const int nh = tl.nhits[t];
      acc = 1ull | ((unsigned long long)nh << 32);
      const unsigned long long key = selKey(nh, tl.chi2[t], (uint32_t)t, wide != 0);
      int kept = 0, first = -1, last = -1;
      const int f = tl.first_row[t], r1 = tl.last_row[t];
      int32_t* row = tl.rowhit + t * tl.n_rows;
      // the kept hits are compacted to the front of the tracklet's own row-hit slice (the write index never passes the
      // read index), so that selectEmit copies `kept` entries instead of walking the rows and the owner keys again
      for (int rb = f & ~3; rb <= r1; rb += 8) {       // eight rows at a time: their owner keys are gathered together
        int32_t c8[8];
        rowHits4(row, tl.n_rows, rb, f, r1, c8);
        if (rb + 4 <= r1) rowHits4(row, tl.n_rows, rb + 4, f, r1, c8 + 4);
        else { c8[4] = c8[5] = c8[6] = c8[7] = -1; }
        // all eight gathers are requested before the first compare (rows without a hit read entry 0 and are masked):
        // behind `c >= 0 &&` each load sat in its own branch and the eight latencies came one after the other
        unsigned long long kk[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) kk[k] = owner_key[c8[k] >= 0 ? c8[k] : 0];
        bool own[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) own[k] = c8[k] >= 0 && kk[k] == key && (!wide || owner_id[c8[k]] == (uint32_t)t);
#pragma unroll
        for (int k = 0; k < 8; ++k)
          if (own[k]) {
            row[f + kept] = c8[k];
            ++kept; if (first < 0) first = rb + k; last = rb + k;
          }
      }
      if (kept >= min_track_hits) {
        sel = 1ull | ((unsigned long long)kept << 32);
        kept_first[t] = first; kept_last[t] = last;
      }
    }
    tsel[t] = sel;
  }
  // block reduction of acc (both halves stay below 2^32 per block)
  for (int d = 16; d > 0; d >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, d);
  __shared__ unsigned long long sm[4];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned long long s = sm[0] + sm[1] + sm[2] + sm[3];
    if (s) {
      atomicAdd((unsigned long long*)(cnt + CNT_N_TRACKLETS), s & 0xffffffffull);
      atomicAdd((unsigned long long*)(cnt + CNT_N_TL_HITS), s >> 32);
    }
  }
}

struct TrackOut {
  int64_t cap_tracks, cap_cl;
  int32_t *tracklet, *sector, *first_row, *last_row, *ncl;
  float *x, *par, *cov, *chi2;
  uint32_t *cl_offset, *cl_index;
};

// per track (tracklet with tsel bit 0): rank k and cluster offset o come from the exclusive scan of tsel.
__global__ void __launch_bounds__(128) selectEmit(TrackletStore tl, const unsigned long long* __restrict__ owner_key,
                                                  const uint32_t* __restrict__ owner_id, int wide,
                                                  const unsigned long long* __restrict__ tsel,
                                                  const unsigned long long* __restrict__ tscan,
                                                  const int32_t* __restrict__ kept_first,
                                                  const int32_t* __restrict__ kept_last,
                                                  const uint32_t* __restrict__ s2o, TrackOut o,
                                                  const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nT = min(cnt[CNT_N_START], tl.capT);
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long sel = t < nT ? tsel[t] : 0ull;
  unsigned long long sc = 0ull;
  bool track = (sel & 1ull) != 0ull;
  if (track) {
    sc = tscan[t];
    if ((int64_t)(sc & 0xffffffffull) >= o.cap_tracks) track = false;
  }
  const int64_t off = (int64_t)(sc >> 32);
  const int kept = (int)(sel >> 32);
  if (track) {        // the per-track values: one lane each (the ranks of a warp's tracks are consecutive)
    const int64_t k = (int64_t)(sc & 0xffffffffull);
    const int64_t capT = tl.capT, capK = o.cap_tracks;
    o.tracklet[k] = (int32_t)t; o.sector[k] = tl.sector[t];
    o.first_row[k] = kept_first[t]; o.last_row[k] = kept_last[t]; o.ncl[k] = kept;
    o.x[k] = tl.x[t]; o.chi2[k] = tl.chi2[t];
#pragma unroll
    for (int i = 0; i < 5; ++i) o.par[i * capK + k] = tl.par[i * capT + t];
#pragma unroll
    for (int i = 0; i < 15; ++i) o.cov[i * capK + k] = tl.cov[i * capT + t];
    o.cl_offset[k] = (uint32_t)off;
  }
  // The cluster lists: the WARP copies the list of each of its tracks together (about one tracklet in twelve is a track:
  // with a thread per track three lanes of a warp were at work, each on its own run of 4-byte loads and stores).  Lane i
  // takes entry i, i + 32, ...: the compacted row hits are read and the indices written as whole lines.
  const int lane = threadIdx.x & 31;
  const int32_t* row = track ? tl.rowhit + t * tl.n_rows + tl.first_row[t] : nullptr;      // compacted by selectCount
  const int nk = track ? (int)max((int64_t)0, min((int64_t)kept, o.cap_cl - off)) : 0;     // entries that fit the output
  unsigned todo = __ballot_sync(0xffffffffu, nk > 0);
  while (todo) {
    const int src = __ffs(todo) - 1;
    todo &= todo - 1;
    const int32_t* r = reinterpret_cast<const int32_t*>(__shfl_sync(0xffffffffu, (unsigned long long)(uintptr_t)row, src));
    const int n = __shfl_sync(0xffffffffu, nk, src);
    const int64_t o0 = __shfl_sync(0xffffffffu, (long long)off, src);
    for (int i = lane; i < n; i += 32) o.cl_index[o0 + i] = s2o[r[i]];
  }
}

// one thread: totals, closing CSR offset, capacity status.
__global__ void finalize(const unsigned long long* __restrict__ sel_total, TrackOut o, int64_t capT,
                         int64_t* __restrict__ cnt) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  if (cnt[CNT_ERROR] != 0) { if (o.cl_offset) o.cl_offset[0] = 0; return; }
  const unsigned long long tot = *sel_total;
  const int64_t ntr = (int64_t)(tot & 0xffffffffull), ncl = (int64_t)(tot >> 32);
  cnt[CNT_N_TRACKS] = ntr;
  cnt[CNT_N_TRK_CL] = ncl;
  o.cl_offset[min(ntr, o.cap_tracks)] = (uint32_t)ncl;
  if (cnt[CNT_N_START] > capT || ntr > o.cap_tracks || ncl > o.cap_cl) cnt[CNT_ERROR] = -4;
}

// ---- optional per-stage exports (parity tests): sorted positions -> global input indices -------------------
__global__ void __launch_bounds__(256) exportLinks(int64_t N, const uint32_t* __restrict__ s2o,
                                                   const int32_t* __restrict__ lup, const int32_t* __restrict__ ldn,
                                                   const int32_t* __restrict__ cup, const int32_t* __restrict__ cdn,
                                                   int32_t* __restrict__ o_ur, int32_t* __restrict__ o_dr,
                                                   int32_t* __restrict__ o_u, int32_t* __restrict__ o_d,
                                                   const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= N) return;
  const uint32_t h = s2o[p];
  int32_t v;
  if (o_ur) { v = lup[p]; o_ur[h] = v >= 0 ? (int32_t)s2o[v] : -1; }
  if (o_dr) { v = ldn[p]; o_dr[h] = v >= 0 ? (int32_t)s2o[v] : -1; }
  if (o_u) { v = cup[p]; o_u[h] = v >= 0 ? (int32_t)s2o[v] : -1; }
  if (o_d) { v = cdn[p]; o_d[h] = v >= 0 ? (int32_t)s2o[v] : -1; }
}

struct TrackletOut {
  uint32_t* start_hits;
  int32_t *status, *nhits, *first_row, *last_row, *rowhit;
  float *x, *par, *cov, *chi2;
};

__global__ void __launch_bounds__(128) exportTracklets(TrackletStore tl, const uint32_t* __restrict__ start_orig,
                                                       const uint32_t* __restrict__ s2o, int n_rows, TrackletOut o,
                                                       const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nT = min(cnt[CNT_N_START], tl.capT);
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nT) return;
  const int64_t capT = tl.capT;
  if (o.start_hits) o.start_hits[t] = start_orig[t];
  const int st = tl.status[t];
  const int f = tl.first_row[t], l = tl.last_row[t];
  if (o.status) o.status[t] = st;
  if (o.nhits) o.nhits[t] = tl.nhits[t];
  if (o.first_row) o.first_row[t] = f;
  if (o.last_row) o.last_row[t] = l;
  const bool has = st != 0 && f >= 0;
  if (o.rowhit)
    for (int r = 0; r < n_rows; ++r) {
      int32_t c = (has && r >= f && r <= l) ? tl.rowhit[t * tl.n_rows + r] : -1;
      o.rowhit[t * n_rows + r] = c >= 0 ? (int32_t)s2o[c] : -1;
    }
  if (o.x) o.x[t] = has ? tl.x[t] : 0.0f;
  if (o.chi2) o.chi2[t] = has ? tl.chi2[t] : 0.0f;
  if (o.par) for (int i = 0; i < 5; ++i) o.par[t * 5 + i] = has ? tl.par[i * capT + t] : 0.0f;
  if (o.cov) for (int i = 0; i < 15; ++i) o.cov[t * 15 + i] = has ? tl.cov[i * capT + t] : 0.0f;
}

}  // namespace tpc
