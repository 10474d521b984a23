// tpc_select.cuh -- a5 tracklet selector (O5; R19..R22, R27) and the optional per-stage exports.
//
// owner(c) = accepted tracklet of highest priority containing c; priority: more hits, then smaller chi2
// (fp32 compare), then smaller tracklet id.  Implemented as atomicMax over a key whose integer order is
// that priority: chi2 >= 0, so its IEEE bit pattern orders like its value.
//   packed key (n_rows <= 255, ids < 2^24):  nhits[63:56] | ~chi2bits[55:24] | ~id[23:0]
//   wide keys  (any id):  pass 1 atomicMax(nhits[63:32] | ~chi2bits[31:0]); pass 2 atomicMin(id) among equals.
#pragma once
#include "tpc_common.cuh"
#ifndef SEL_NB
#define SEL_NB 3                      // selectCount: blocks of 32 rows a warp takes per trip (their owner keys gathered together;
                                      // 1 / 2 / 3 / 4: 2.12 / 1.69 / 1.65 / 1.78 ms)
#endif

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
  const bool accepted = t < nT && tl.status[t] == 2;
  unsigned long long key = 0ull;
  int f = 0, r1 = -1;
  if (accepted) {
    const int nh = tl.nhits[t];
    acc = 1ull | ((unsigned long long)nh << 32);
    key = selKey(nh, tl.chi2[t], (uint32_t)t, wide != 0);
    f = tl.first_row[t]; r1 = tl.last_row[t];
  }
  // The WARP walks the rows of each of its accepted tracklets together: lane i takes rows f + i, f + i + 32, ... of a trip
  // (whole lines of the row-hit slice, 32 x SEL_NB owner keys gathered at once), the kept hits are compacted to the front of the
  // slice by ballot and prefix count -- the write index never passes the rows read -- so that selectEmit only copies.
  // (A thread per tracklet walked its own slice eight rows at a time: 7.7 of 32 lanes, 1.4e9 warp instructions.)
  const int lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  int kept = 0, first = -1, last = -1;
  unsigned todo = __ballot_sync(0xffffffffu, accepted);
  while (todo) {
    const int src = __ffs(todo) - 1;
    todo &= todo - 1;
    const unsigned long long k = __shfl_sync(0xffffffffu, key, src);
    const int ff = __shfl_sync(0xffffffffu, f, src), rr = __shfl_sync(0xffffffffu, r1, src);
    const uint32_t tt = (uint32_t)(t - lane + src);
    int32_t* row = tl.rowhit + (int64_t)tt * tl.n_rows;
    int kk = 0, fi = -1, la = -1;                 // the same in every lane
    for (int rb = ff; rb <= rr; rb += 32 * SEL_NB) {
      int32_t c[SEL_NB];
      unsigned long long kq[SEL_NB];
      unsigned m[SEL_NB];
#pragma unroll
      for (int q = 0; q < SEL_NB; ++q) { const int r = rb + 32 * q + lane; c[q] = r <= rr ? row[r] : -1; }
#pragma unroll
      for (int q = 0; q < SEL_NB; ++q) kq[q] = owner_key[c[q] >= 0 ? c[q] : 0];
#pragma unroll
      for (int q = 0; q < SEL_NB; ++q) {
        const bool own = c[q] >= 0 && kq[q] == k && (!wide || owner_id[c[q]] == tt);
        m[q] = __ballot_sync(0xffffffffu, own);
        if (own) row[ff + kk + __popc(m[q] & lt)] = c[q];
        if (m[q]) {
          if (fi < 0) fi = rb + 32 * q + __ffs(m[q]) - 1;
          la = rb + 32 * q + 31 - __clz(m[q]);
          kk += __popc(m[q]);
        }
      }
    }
    if (lane == src) { kept = kk; first = fi; last = la; }
  }
  if (t < nT) {
    unsigned long long sel = 0;
    if (accepted && kept >= min_track_hits) {
      sel = 1ull | ((unsigned long long)kept << 32);
      kept_first[t] = first; kept_last[t] = last;
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
