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

#ifndef TC_THREADS_
#define TC_THREADS_ 128
#endif
constexpr int TC_THREADS = TC_THREADS_;
#ifndef TC_MIN_BLOCKS
#define TC_MIN_BLOCKS 5
#endif
#ifndef TC_MB_UP
#define TC_MB_UP TC_MIN_BLOCKS          // resident CTAs per SM the three passes are compiled for (register budget)
#endif
#ifndef TC_MB_SPAN
#define TC_MB_SPAN TC_MIN_BLOCKS
#endif
#ifndef TC_MB_EXT
#define TC_MB_EXT TC_MIN_BLOCKS
#endif
constexpr int MAX_ROWS = 256;
#ifndef TC_HEADS
#define TC_HEADS 6                  // candidates per cell row loaded and evaluated without a loop
#endif

// Search (O4): nearest cluster of the bucket inside the road around the predicted (y,z); key (d2, orig index).
// Split in two so that the first grid loads are in flight while Propagate finishes the covariance transport:
// searchBegin (called from Propagate's hook) computes the road and the cell window and loads the cell ranges
// of the first two cell rows; searchFinish scans the candidates.
struct SearchPre {
  float yp, zp, ry, rz;
  int bz0, bz1, ny, span;
  const uint32_t* cs;        // cell_start + cell_base + by0
  uint32_t kA0, kA1, kB0, kB1;
};

__device__ __forceinline__ void searchBegin(SearchPre& sp, float yp, float zp, float c00, float c11, const GridDesc& G,
                                            const uint32_t* __restrict__ cell_start, const DevParams& P) {
  float ry = P.road_sigma * sqrtf(c00 + P.err2_y);
  float rz = P.road_sigma * sqrtf(c11 + P.err2_z);
  if (!(ry >= P.road_min)) ry = P.road_min;
  if (ry > P.road_max) ry = P.road_max;
  if (!(rz >= P.road_min)) rz = P.road_min;
  if (rz > P.road_max) rz = P.road_max;
  const float sy = 1e-5f * (fabsf(yp) + ry) + 1e-6f;      // superset slack, see forWindow
  const float sz = 1e-5f * (fabsf(zp) + rz) + 1e-6f;
  const int by0 = cellCoord((yp - ry) - sy, G.y0, G.inv_e, G.ny);
  const int by1 = cellCoord((yp + ry) + sy, G.y0, G.inv_e, G.ny);
  sp.bz0 = cellCoord((zp - rz) - sz, G.z0, G.inv_e, G.nz);
  sp.bz1 = cellCoord((zp + rz) + sz, G.z0, G.inv_e, G.nz);
  sp.yp = yp; sp.zp = zp; sp.ry = ry; sp.rz = rz;
  sp.ny = G.ny; sp.span = by1 - by0 + 1;
  sp.cs = cell_start + G.cell_base + by0;
  const uint32_t* rA = sp.cs + sp.bz0 * G.ny;
  const uint32_t* rB = sp.cs + min(sp.bz0 + 1, sp.bz1) * G.ny;
  sp.kA0 = __ldg(rA); sp.kA1 = __ldg(rA + sp.span);
  sp.kB0 = __ldg(rB); sp.kB1 = __ldg(rB + sp.span);
}

// Exact re-scan of a window with the full key (d2, original index): only after the fast scan saw two candidates
// at exactly the same distance (duplicated clusters, R6).
__device__ __noinline__ int32_t searchExact(const SearchPre& sp, const float2* __restrict__ syz,
                                            const uint32_t* __restrict__ s2o, float* ym, float* zm) {
  int32_t best = -1;
  float bestd = 0.0f, by = 0.0f, bz = 0.0f;
  for (int r = sp.bz0; r <= sp.bz1; ++r) {
    const uint32_t* row = sp.cs + r * sp.ny;
    const uint32_t k1 = __ldg(row + sp.span);
    for (uint32_t k = __ldg(row); k < k1; ++k) {
      const float2 c = __ldg(syz + k);
      if (fabsf(c.x - sp.yp) <= sp.ry && fabsf(c.y - sp.zp) <= sp.rz) {
        const float dy = c.x - sp.yp, dz = c.y - sp.zp;
        const float d2 = dy * dy + dz * dz;
        if (best < 0 || d2 < bestd || (d2 == bestd && __ldg(s2o + k) < __ldg(s2o + best))) {
          best = (int32_t)k; bestd = d2; by = c.x; bz = c.y;
        }
      }
    }
  }
  *ym = by; *zm = bz;
  return best;
}

// returns the sorted position of the best cluster or -1; its coordinates in (ym, zm).
// The heads of the two prefetched cell rows (up to TC_HEADS + TC_HEADS candidates, every load in flight before the first test:
// one memory latency per search instead of one per candidate) are evaluated without branches; unused slots hold
// a point outside every window.  Longer rows and further cell rows are scanned by loops.
__device__ __forceinline__ int32_t searchFinish(const SearchPre& sp, const float2* __restrict__ syz,
                                                const uint32_t* __restrict__ s2o, float& ym, float& zm) {
  const float yp = sp.yp, zp = sp.zp, ry = sp.ry, rz = sp.rz;
  const uint32_t nA = sp.kA1 - sp.kA0;
  const uint32_t nB = sp.bz1 > sp.bz0 ? sp.kB1 - sp.kB0 : 0u;
  const float2 far = make_float2(3.0e38f, 3.0e38f);
  float2 ca[TC_HEADS], cb[TC_HEADS];
#pragma unroll
  for (int i = 0; i < TC_HEADS; ++i) ca[i] = i < nA ? __ldg(syz + sp.kA0 + i) : far;
#pragma unroll
  for (int i = 0; i < TC_HEADS; ++i) cb[i] = i < nB ? __ldg(syz + sp.kB0 + i) : far;
  float bestd = __int_as_float(0x7f800000);     // d2 of a candidate inside the road is finite
  int32_t best = -1;
  bool tie = false;
  auto eval = [&](const float2 c, uint32_t k) {
    const bool in = fabsf(c.x - yp) <= ry && fabsf(c.y - zp) <= rz;
    const float dy = c.x - yp, dz = c.y - zp;
    const float d2 = dy * dy + dz * dz;
    tie = tie || (in && d2 == bestd);
    const bool better = in && d2 < bestd;
    best = better ? (int32_t)k : best;
    bestd = better ? d2 : bestd;
    ym = better ? c.x : ym;
    zm = better ? c.y : zm;
  };
#pragma unroll
  for (int i = 0; i < TC_HEADS; ++i) eval(ca[i], sp.kA0 + i);
#pragma unroll
  for (int i = 0; i < TC_HEADS; ++i) eval(cb[i], sp.kB0 + i);
  auto scan = [&](uint32_t k0, uint32_t k1) {      // two independent loads per trip
    for (uint32_t k = k0; k < k1; k += 2) {
      const bool two = k + 1 < k1;
      const float2 a = __ldg(syz + k);
      const float2 c = two ? __ldg(syz + k + 1) : far;
      eval(a, k);
      eval(c, k + 1);
    }
  };
  if (nA > TC_HEADS) scan(sp.kA0 + TC_HEADS, sp.kA1);
  if (nB > TC_HEADS) scan(sp.kB0 + TC_HEADS, sp.kB1);
  for (int bz = sp.bz0 + 2; bz <= sp.bz1; ++bz) {   // roads wider than two cell rows: rare
    const uint32_t* r = sp.cs + bz * sp.ny;
    scan(__ldg(r), __ldg(r + sp.span));
  }
  if (tie) {     // the out-of-line re-scan gets copies: `sp`, `ym`, `zm` themselves must never have their address taken,
                 // or they live in local memory and the store of the cell ranges waits for their loads right in searchBegin
    const SearchPre cp = sp;
    float ey = 0.0f, ez = 0.0f;
    best = searchExact(cp, syz, s2o, &ey, &ez);
    ym = ey; zm = ez;
  }
  return best;
}

// One long seed in the constructor's work list (32 bytes, written by seedPrepare).
struct SeedRec {
  uint32_t t, h0;        // tracklet id, sorted position of the start hit
  int32_t h1;            // first link
  uint32_t b0r0;         // sector << 22 | bucket << 8 | row of the start hit
  float y0, z0, s0, t0;  // O4 step 1: coordinates of h0, and sin phi and dz/ds of the first link (computed by seedPrepare)
};

// One thread per start hit, before the constructor: bucket of the seed, length of its link chain.  Chains shorter
// than min_chain_hits can only end as "discarded in the chain fit" (O4 step 2): they are fitted right here (the
// hit count of a discarded tracklet is part of the per-stage output) and never reach the persistent kernel;
// the others are appended to the constructor's work list.  At high occupancy most start hits are such stubs.
__global__ void __launch_bounds__(128) seedPrepare(const uint32_t* __restrict__ off, DevParams P, RowTables T,
                                                   const float2* __restrict__ syz, const int32_t* __restrict__ cup,
                                                   const uint32_t* __restrict__ start_pos, SeedRec* __restrict__ work,
                                                   TrackletStore out, int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nT = min(cnt[CNT_N_START], out.capT);
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nT) return;
  const uint32_t h0 = start_pos[t];
  const int b0 = bucketOf(off, P.n_buckets, h0);
  const int R = P.n_rows;
  const int r0 = b0 % R;
  out.sector[t] = b0 / R;
  int len = 1;
  for (int32_t h = cup[h0]; h != -1 && len < P.min_chain_hits; h = cup[h]) ++len;
  if (len >= P.min_chain_hits) {
    const unsigned long long j = atomicAdd((unsigned long long*)(cnt + CNT_N_LONG), 1ull);
    const int32_t h1 = cup[h0];
    const float2 a = syz[h0], c = syz[h1];
    // O4 step 1 here, at full lanes, instead of at the 5 lanes of the constructor's seed fetch
    const float dx = T.row_x[T.up_row[r0]] - T.row_x[r0], dy = c.x - a.x, dz = c.y - a.y;
    const float L = sqrtf(dx * dx + dy * dy);
    uint4* q = reinterpret_cast<uint4*>(work + j);
    q[0] = make_uint4((uint32_t)t, h0, (uint32_t)h1, ((uint32_t)(b0 / R) << 22) | ((uint32_t)b0 << 8) | (uint32_t)r0);
    q[1] = make_uint4(__float_as_uint(a.x), __float_as_uint(a.y), __float_as_uint(dy / L), __float_as_uint(dz / L));
    return;
  }
  // short chain: O4 steps 1-2 on its len-1 links; the result is always status 0, nhits = hits fitted
  int r = T.up_row[r0];
  int32_t h = cup[h0];
  KFState S;
  {
    const float2 a = syz[h0], c = syz[h];
    S.x = T.row_x[r0]; S.y = a.x; S.z = a.y;
    const float dx = T.row_x[r] - T.row_x[r0], dy = c.x - a.x, dz = c.y - a.y;
    const float L = sqrtf(dx * dx + dy * dy);
    S.s = dy / L; S.t = dz / L; S.q = 0.0f;
  }
  kfSetDiag(S, P.err2_y, P.err2_z, P);
  S.chi2 = 0.0f;
  int nhits = 1;
  while (h != -1) {
    if (!kfPropagate(S, T.row_x[r], P, [](float, float, float, float) {})) break;
    const float2 c = syz[h];
    if (!kfUpdate(S, c.x, c.y, P)) break;
    ++nhits;
    h = cup[h];
    r = T.up_row[r];
  }
  out.status[t] = 0; out.nhits[t] = nhits; out.first_row[t] = -1; out.last_row[t] = -1;
}

// ---- the three passes of O4 as three persistent kernels -------------------------------------------------------------
// Every lane owns one seed at a time and fetches the next one from a global counter as soon as its seed is finished
// ("lane refill"), so a warp stays full although seeds need between 1 and ~150 steps per pass.  A step is
//     Propagate -> candidate (link | known hit | Search) -> Update -> bookkeeping.
// The passes run as SEPARATE kernels so that the lanes of a warp do the same kind of step:
//   constructUp        chain fit (links) and up extrapolation (a Search per row)          -> TurnRec  (32 bytes per seed)
//   constructDown<0>   down pass over the span [r0, top]: the hits are known, Searches only on the rare gap rows
//                                                                                         -> DownRec (112 bytes per seed)
//   constructDown<1>   down pass below r0: a Search per row, miss counting                 -> the tracklet
// In one kernel (round 1) the Search code ran whenever any lane of the warp wanted it, at 19.6 of 32 lanes, and the
// phase bookkeeping at 12.3 lanes.  The hand-off records cost 0.3 GB of writes and reads per event, the time of 0.1 ms.
// The order of the floating-point operations of a seed is exactly the sequential algorithm's; the turn (O4 step 4) keeps
// only the parameters, so a TurnRec carries five floats.
// Loads are software-pipelined around the arithmetic: the hit of a step (link or known row hit) is fetched one step
// ahead, its coordinates and the row's grid descriptor are requested before Propagate, the cell ranges of a search from
// inside Propagate.

constexpr uint32_t REC_NONE = 0xFFFFFFFFu;

struct TurnRec {           // state of a seed at the turn (O4 step 4)
  uint32_t t;              // tracklet id; REC_NONE = the seed ended in the chain fit
  int32_t last_c;          // the hit on the top row
  float y, z, s, tt, q;    // parameters at plane row_x[rx]
  uint32_t rows;           // r0 | top row << 8 | rx << 16 | TURN_HAS_GAP | sector << 25
};
constexpr uint32_t TURN_HAS_GAP = 1u << 24;     // some live row inside (r0, top) has no hit: the span pass searches there
constexpr int TURN_SECTOR_SHIFT = 25;           // the sector rides along (< 64): no load of out.sector in the span pass
static_assert(sizeof(TurnRec) == 32, "TurnRec is two 16-byte words");

// state of a seed after the Update on its start row r0, going down: t, rows (r0 | top << 8), nhits, pad, then
// y z s t q, c00..c44, chi2 (21 floats) and 3 floats of padding: seven 16-byte words
constexpr int DOWNREC_WORDS = 28;

struct RowSmem {
  float sx[MAX_ROWS];
  int16_t sup[MAX_ROWS];          // up_row (R2)
  int16_t snu[MAX_ROWS];          // next live row above (n_rows if none)
  int16_t snd[MAX_ROWS];          // next live row below (-1 if none)
};

__device__ __forceinline__ void rowSmemFill(RowSmem& rs, const RowTables& T, int R) {
  for (int i = threadIdx.x; i < R; i += blockDim.x) {
    rs.sx[i] = T.row_x[i]; rs.sup[i] = T.up_row[i];
    int u = i + 1, d = i - 1;
    while (u < R && T.dead[u]) ++u;
    while (d >= 0 && T.dead[d]) --d;
    rs.snu[i] = (int16_t)u; rs.snd[i] = (int16_t)d;
  }
  __syncthreads();
}

#define TC_SNAP_STORE(snap, tid, S)                                                                                   \
  do {                                                                                                                \
    snap[0][tid] = S.x; snap[1][tid] = S.y; snap[2][tid] = S.z; snap[3][tid] = S.s; snap[4][tid] = S.t;               \
    snap[5][tid] = S.q; snap[6][tid] = S.chi2; snap[7][tid] = S.c00; snap[8][tid] = S.c10; snap[9][tid] = S.c11;      \
    snap[10][tid] = S.c20; snap[11][tid] = S.c21; snap[12][tid] = S.c22; snap[13][tid] = S.c30;                       \
    snap[14][tid] = S.c31; snap[15][tid] = S.c32; snap[16][tid] = S.c33; snap[17][tid] = S.c40;                       \
    snap[18][tid] = S.c41; snap[19][tid] = S.c42; snap[20][tid] = S.c43; snap[21][tid] = S.c44;                       \
  } while (0)

// O4 step 6: the tracklet is the last snapshot of the down pass (state at the innermost attached row)
__device__ __forceinline__ void writeTracklet(const TrackletStore& out, const DevParams& P, uint32_t t, int nhits,
                                              int snap_row, int rtop, float (*snap)[TC_THREADS], int tid) {
  if (snap_row < 0) {
    out.status[t] = 1; out.nhits[t] = 0; out.first_row[t] = -1; out.last_row[t] = -1;
    return;
  }
  const int64_t capT = out.capT;
  out.status[t] = nhits >= P.min_tracklet_hits ? 2 : 1;
  out.nhits[t] = nhits; out.first_row[t] = snap_row; out.last_row[t] = rtop;
  out.x[t] = snap[0][tid]; out.chi2[t] = snap[6][tid];
#pragma unroll
  for (int i = 0; i < 5; ++i) out.par[i * capT + t] = snap[1 + i][tid];
#pragma unroll
  for (int i = 0; i < 15; ++i) out.cov[i * capT + t] = snap[7 + i][tid];
}

// Work distribution of the persistent passes.  A lane that has finished its seed needs the next index of the pass's list.
// Drawn per lane from a global counter, that is an atomic round trip to the L2, then the load of the record, then -- in
// the down passes, before the records carried the sector -- the load of the tracklet's sector: dependent memory latencies
// during which the other lanes of the warp stand still (11 % of the stall samples of the passes, profiles/r2d).  With
// drawIndex a warp draws TC_CHUNK consecutive indices with ONE atomic, keeps the chunk in shared memory and hands its
// indices out to the lanes that ask (in lane order, by ballot); the records of the chunk are requested into the L2 when
// the chunk is drawn.  Used by the search-free span instance only (see constructDown).
#ifndef TC_CHUNK_
#define TC_CHUNK_ 32
#endif
#ifndef TC_PF_AHEAD
#define TC_PF_AHEAD 2048            // passes with the global counter: the record this many draws ahead is requested into the L2
                                    // by the lane that draws now (records come from DRAM: written by the pass before, 0.3-0.5 GB;
                                    // up pass 7.84 -> 7.74 ms, pass below r0 10.66 -> 10.56 ms; 1024 and 4096 give the same)
#endif
constexpr uint32_t TC_CHUNK = TC_CHUNK_;

__device__ __forceinline__ void prefetchL2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// Warp-synchronous (all 32 lanes call it together).  Lanes with `want` get the next indices of the warp's chunk in lane
// order; returns true and the index in j for those served.  A lane that wants and is not served (the chunk ran out
// in front of it) asks again: the next call draws a new chunk.  The indices may lie beyond the end of the list (the
// caller checks); `rec` / `rec_bytes` / `n_rec` describe the record array to prefetch (rec may be NULL).
__device__ __forceinline__ bool drawIndex(bool want, unsigned long long* __restrict__ work, volatile uint32_t* w_next,
                                          volatile uint32_t* w_end, const void* rec, uint32_t rec_bytes, int64_t n_rec,
                                          uint32_t& j) {
  const unsigned need = __ballot_sync(0xffffffffu, want);
  const uint32_t lane = threadIdx.x & 31u;
  uint32_t nxt = *w_next, end = *w_end;
  if (nxt == end) {                    // uniform over the warp: the chunk is used up (or none drawn yet)
    uint32_t base = 0;
    if (lane == 0) base = (uint32_t)atomicAdd(work, (unsigned long long)TC_CHUNK);
    base = __shfl_sync(0xffffffffu, base, 0);
    nxt = base; end = base + TC_CHUNK;
    if (lane == 0) *w_end = end;
    if (rec) {
      const int64_t last = min((int64_t)end, n_rec);
      const char* a = reinterpret_cast<const char*>(rec) + (int64_t)base * rec_bytes;
      const char* e = reinterpret_cast<const char*>(rec) + last * rec_bytes;
      for (const char* q = a + lane * 128; q < e; q += 32 * 128) prefetchL2(q);
    }
  }
  const uint32_t avail = end - nxt;
  const uint32_t rank = __popc(need & ((1u << lane) - 1u));
  const uint32_t take = min((uint32_t)__popc(need), avail);
  __syncwarp();                        // every lane has read w_next
  if (lane == 0) *w_next = nxt + take;
  __syncwarp();
  j = nxt + rank;
  return want && rank < avail;
}

// ---- pass 1: chain fit (O4 step 2) and up extrapolation (step 3) ---------------------------------------------------
__global__ void __launch_bounds__(TC_THREADS, TC_MB_UP) constructUp(
    DevParams P, RowTables T, const GridDesc* __restrict__ desc, const uint32_t* __restrict__ cell_start,
    const float2* __restrict__ syz, const uint32_t* __restrict__ s2o, const int32_t* __restrict__ cup,
    const SeedRec* __restrict__ work_list, TurnRec* __restrict__ turn_list, TrackletStore out, int64_t* __restrict__ cnt) {
  __shared__ RowSmem rs;
  // per-lane bookkeeping that is read once per step or less lives in shared memory (volatile: re-read where used):
  // in registers it pushed the kernel over its budget and the spilled bucket base sat on the path to every grid load
  __shared__ volatile uint32_t s_t[TC_THREADS];       // tracklet id
  __shared__ volatile uint32_t s_j[TC_THREADS];       // index of the seed in the work list
  __shared__ volatile int s_bsec[TC_THREADS];         // first bucket of the seed's sector
  __shared__ volatile int16_t s_rc[TC_THREADS];       // row of the last Propagate
  __shared__ volatile uint8_t s_sec[TC_THREADS];      // sector of the seed
  if (cnt[CNT_ERROR] != 0) return;
  const int R = P.n_rows;
  const int tid = threadIdx.x;
  rowSmemFill(rs, T, R);
  const int64_t nW = cnt[CNT_N_LONG];            // seeds on the work list (seedPrepare)
  unsigned long long* work = (unsigned long long*)(cnt + CNT_WORK);

  KFState S;
  int phase = -1;                 // -1 wants a seed, -2 no seeds left, 0 chain fit, 1 up extrapolation
  int32_t* rowhit = nullptr;      // this tracklet's [n_rows] slice
  int r0 = 0, rn = 0, lastw = 0, nhits = 0, miss = 0;
  int32_t c_cur = -1;             // hit of the coming step if known (link), else -1 = search
  int32_t last_c = -1;            // last recorded hit (the hit on row lastw)
  // a live row without a hit (a miss, or a refused Update) that a later hit closes in is a gap row of the span: the span
  // pass must search there.  Seeds without one go to the search-free span kernel.
  bool open_miss = false, has_gap = false;

  for (;;) {
    if (phase == -1) {            // ---- fetch and initialise the next seed (O4 step 1) ----
      const int64_t j = (int64_t)atomicAdd(work, 1ull);
      if (j >= nW) {
        phase = -2;
      } else {
        const uint4* rp = reinterpret_cast<const uint4*>(work_list + j);
        const uint4 a = __ldg(rp), b = __ldg(rp + 1);
#if TC_PF_AHEAD
        if (j + TC_PF_AHEAD < nW) prefetchL2(work_list + j + TC_PF_AHEAD);     // for the lane that will draw it
#endif
        const uint32_t t = a.x;
        s_t[tid] = t; s_j[tid] = (uint32_t)j;
        const uint32_t h0 = a.y;
        c_cur = (int32_t)a.z;
        r0 = (int)(a.w & 0xffu);
        s_bsec[tid] = (int)((a.w >> 8) & 0x3fffu) - r0;
        s_sec[tid] = (uint8_t)(a.w >> 22);
        rowhit = out.rowhit + (int64_t)t * R;
        rn = rs.sup[r0];
        const float y0 = __uint_as_float(b.x), z0 = __uint_as_float(b.y);
        S.x = rs.sx[r0]; S.y = y0; S.z = z0;
        S.s = __uint_as_float(b.z); S.t = __uint_as_float(b.w); S.q = 0.0f;
        kfSetDiag(S, P.err2_y, P.err2_z, P);
        S.chi2 = 0.0f;
        rowhit[r0] = (int32_t)h0;
        last_c = (int32_t)h0;
        nhits = 1; s_rc[tid] = (int16_t)r0; lastw = r0; miss = 0;
        open_miss = false; has_gap = false;
        phase = 0;
      }
    }
    if (__all_sync(0xffffffffu, phase == -2)) break;

    // ---- one step: early loads -> Propagate (search loads issued inside) -> candidate -> Update ----
    const bool act = phase >= 0;
    float ym = 0.0f, zm = 0.0f;
    float2 mk = make_float2(0.0f, 0.0f);         // coordinates of the link: consumed only at the Update
    int32_t hnext = -1;
    // the grid descriptor of the row is loaded by every lane (a conditional struct assignment would make the compiler
    // wait for the load right here, to merge it with the "not loaded" value)
    const GridDesc G = desc[act ? s_bsec[tid] + rn : 0];
    if (act && c_cur >= 0) {
      mk = __ldg(syz + c_cur);
      hnext = __ldg(cup + c_cur);
    }
    SearchPre sp;
    const bool want_search = act && c_cur < 0;
    const bool okp = act && kfPropagate(S, rs.sx[act ? rn : 0], P, [&](float y1, float z1, float c00, float c11) {
      if (want_search) searchBegin(sp, y1, z1, c00, c11, G, cell_start, P);
    });
    int32_t c = c_cur;
    if (okp && c < 0) c = searchFinish(sp, syz, s2o, ym, zm);
    if (c_cur >= 0) { ym = mk.x; zm = mk.y; }
    bool oku = false;
    if (okp && c >= 0) oku = kfUpdate(S, ym, zm, P);
    if (!act) continue;

    // ---- bookkeeping and phase transitions ----
    bool end_phase = !okp || (c >= 0 && !oku);       // Propagate or Update refused: the pass ends here
    bool turn = false;
    const int rb = rn;                               // the row of this step
    if (okp) { rowhit[rb] = oku ? c : -1; s_rc[tid] = (int16_t)rb; }    // rows beyond the final first/last row are never read
    if (okp) { has_gap = has_gap || (oku && open_miss); open_miss = open_miss || !oku; }
    if (phase == 0) {
      if (oku) {
        lastw = rb; last_c = c; ++nhits;
        c_cur = hnext;
        rn = rs.sup[rb];
        if (hnext == -1) end_phase = true;
      }
      if (end_phase) {
        if (nhits < P.min_chain_hits) {
          const uint32_t t = s_t[tid];
          out.status[t] = 0; out.nhits[t] = nhits; out.first_row[t] = -1; out.last_row[t] = -1;
          turn_list[s_j[tid]].t = REC_NONE;
          phase = -1;
        } else {
          phase = 1; miss = 0; c_cur = -1;
          rn = rs.snu[s_rc[tid]];
          if (rn >= R) turn = true;
        }
      }
    } else {
      if (oku) {
        lastw = rb; last_c = c; ++nhits; miss = 0;
      } else if (!end_phase) {
        if (++miss > P.max_row_gap) end_phase = true;
      }
      if (!end_phase) {
        rn = rs.snu[rb];
        if (rn >= R) end_phase = true;
      }
      if (end_phase) turn = true;
    }
    if (turn) {                   // O4 step 4 happens in the next kernel: hand the parameters over
      uint4* q = reinterpret_cast<uint4*>(turn_list + s_j[tid]);
      q[0] = make_uint4(s_t[tid], (uint32_t)last_c, __float_as_uint(S.y), __float_as_uint(S.z));
      q[1] = make_uint4(__float_as_uint(S.s), __float_as_uint(S.t), __float_as_uint(S.q),
                        (uint32_t)r0 | ((uint32_t)lastw << 8) | (((uint32_t)(uint16_t)s_rc[tid] & 0xffu) << 16) |
                            (has_gap ? TURN_HAS_GAP : 0u) | ((uint32_t)s_sec[tid] << TURN_SECTOR_SHIFT));
      phase = -1;
    } else if (phase >= 0 && P.any_dead) {      // dead rows stepped over (R23) hold no hit
      const int lo = min(rb, rn), hi = max(rb, rn);
      if (hi - lo > 1)
        for (int g = lo + 1; g < hi; ++g) rowhit[g] = -1;
    }
  }
}

// The seeds whose span has a gap row, as a dense list of work-list indices in ascending order inside every block of 1024
// (the blocks append their runs with one atomic each): the gap instance of the span pass takes its seeds from it.
// The order matters: seeds that are neighbours in the work list are neighbours in the detector, and the passes live on
// the L2 hits of their grid and cluster gathers (a list in completion order cost the last pass 24 GB of DRAM reads
// instead of 9 GB).
__global__ void __launch_bounds__(1024) gapListBuild(const TurnRec* __restrict__ turn_list, uint32_t* __restrict__ gap_idx,
                                                     int64_t* __restrict__ cnt) {
  __shared__ uint32_t sm[33];
  __shared__ uint32_t s_base;
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nW = cnt[CNT_N_LONG];
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if ((int64_t)blockIdx.x * blockDim.x >= nW) return;
  const bool gap = j < nW && turn_list[j].t != REC_NONE && (turn_list[j].rows & TURN_HAS_GAP) != 0u;
  uint32_t total;
  const uint32_t pre = blockExclusiveScan(gap ? 1u : 0u, sm, &total);
  if (threadIdx.x == 0) s_base = total ? (uint32_t)atomicAdd((unsigned long long*)(cnt + CNT_N_GAP), (unsigned long long)total) : 0u;
  __syncthreads();
  if (gap) gap_idx[s_base + pre] = (uint32_t)j;
}

// ---- passes 2 and 3: the down pass (O4 steps 4-6), over the span (EXT = 0) and below the start row (EXT = 1) -----------
// GAP (span pass only): 1 = the seeds whose span has gap rows (taken from gap_idx), with the Search code; 0 = the others
// (the whole list, skipping the seeds of the other kind), without it.  In one kernel the whole warp issued the search code
// on nearly every step for the 1.5 lanes that stood on a gap row: 20 % of the span pass's instructions.
template <int EXT, int GAP>
__global__ void __launch_bounds__(TC_THREADS, EXT ? TC_MB_EXT : TC_MB_SPAN) constructDown(
    DevParams P, RowTables T, const GridDesc* __restrict__ desc, const uint32_t* __restrict__ cell_start,
    const float2* __restrict__ syz, const uint32_t* __restrict__ s2o, const TurnRec* __restrict__ turn_list,
    const uint32_t* gap_idx, uint4* __restrict__ down_list, TrackletStore out, int64_t* __restrict__ cnt) {
  uint32_t* gap_idx_out = const_cast<uint32_t*>(gap_idx);       // written by the search-free instance only (refused seeds)
  __shared__ RowSmem rs;
  __shared__ float snap[22][TC_THREADS];     // state after the last Update (O4 step 5)
  __shared__ volatile uint32_t s_t[TC_THREADS];
  __shared__ volatile uint32_t s_j[TC_THREADS];
  __shared__ volatile int s_bsec[TC_THREADS];
  __shared__ volatile int16_t s_rtop[TC_THREADS];
  __shared__ volatile uint32_t s_wn[TC_THREADS / 32], s_we[TC_THREADS / 32];      // the warp's chunk of work indices
  if (cnt[CNT_ERROR] != 0) return;
  const int R = P.n_rows;
  const int tid = threadIdx.x;
  if ((tid & 31) == 0) { s_wn[tid >> 5] = 0; s_we[tid >> 5] = 0; }
  rowSmemFill(rs, T, R);
  const int64_t nW = cnt[(!EXT && GAP) ? CNT_N_GAP : CNT_N_LONG];
  unsigned long long* work = (unsigned long long*)(cnt + (EXT ? CNT_WORK3 : GAP ? CNT_WORK4 : CNT_WORK2));

  KFState S;
  int phase = -1;                 // -1 wants a seed, -2 no seeds left, 2 down pass
  int32_t* rowhit = nullptr;
  int r0 = 0, rn = 0, nhits = 0, miss = 0, snap_row = -1;
  int32_t c_cur = -1;             // hit of the coming step if known (row hit), else -1 = search
  // row hit of the step after, loaded one step ahead.  Kept as (raw value, valid) and merged with -1 only when it
  // becomes c_cur: a select right behind the load would wait for the load and undo the pipelining.
  int32_t nx_raw = -1;
  bool nx_ok = false;

  for (;;) {
    // The search-free span instance draws its indices a chunk per warp (see drawIndex); the instances that search keep
    // the one global counter: with chunks their seeds in flight spread over more rows of the detector and the gathers of
    // the searches miss the L2 (measured with chunks of 64: L2 hit rate of the pass below r0 67 -> 46 %, DRAM reads
    // 9.4 -> 27 GB, 10.7 -> 13.0 ms; the up pass 7.8 -> 8.8 ms; even chunks of 4 cost 6 %).
    constexpr bool CHUNKED = !EXT && !GAP;
    while (CHUNKED ? __any_sync(0xffffffffu, phase == -1) : phase == -1) {         // ---- fetch the next seed that is still alive ----
      int64_t j;
      if (CHUNKED) {
        uint32_t jw;
        if (!drawIndex(phase == -1, work, &s_wn[tid >> 5], &s_we[tid >> 5], turn_list, (uint32_t)sizeof(TurnRec), nW, jw)) continue;
        j = (int64_t)jw;
      } else {
        j = (int64_t)atomicAdd(work, 1ull);
      }
      if (j >= nW) { phase = -2; if (CHUNKED) continue; else break; }
      if (!EXT) {
        if (GAP) j = (int64_t)gap_idx[j];
        const uint4* rp = reinterpret_cast<const uint4*>(turn_list + j);
        const uint4 a = __ldg(rp), b = __ldg(rp + 1);
        if (!GAP) {
          if (a.x == REC_NONE) { down_list[j * (DOWNREC_WORDS / 4)].x = REC_NONE; continue; }
          if ((b.w & TURN_HAS_GAP) != 0u) continue;                     // the gap instance's seed
        }
        const uint32_t t = a.x;
        s_t[tid] = t; s_j[tid] = (uint32_t)j;
        r0 = (int)(b.w & 0xffu);
        const int rtop = (int)((b.w >> 8) & 0xffu), rx = (int)((b.w >> 16) & 0xffu);
        s_rtop[tid] = (int16_t)rtop;
        s_bsec[tid] = (int)(b.w >> TURN_SECTOR_SHIFT) * R;
        rowhit = out.rowhit + (int64_t)t * R;
        // O4 step 4: diffuse covariance, parameters kept (R17); the down pass starts at the top row
        S.x = rs.sx[rx]; S.y = __uint_as_float(a.z); S.z = __uint_as_float(a.w);
        S.s = __uint_as_float(b.x); S.t = __uint_as_float(b.y); S.q = __uint_as_float(b.z);
        kfSetDiag(S, P.turn_var_scale * P.err2_y, P.turn_var_scale * P.err2_z, P);
        S.chi2 = 0.0f;
        rn = rtop; miss = 0; nhits = 0; snap_row = -1;
        c_cur = (int32_t)a.y;       // the hit on the top row
        const int r2 = rs.snd[rn];
        nx_ok = r2 >= r0;
        if (nx_ok) nx_raw = rowhit[r2];
        phase = 2;
      } else {
        const uint4* rp = down_list + j * (DOWNREC_WORDS / 4);
#if TC_PF_AHEAD
        if (j + TC_PF_AHEAD < nW) {
          prefetchL2(down_list + (j + TC_PF_AHEAD) * (DOWNREC_WORDS / 4));
          prefetchL2(down_list + (j + TC_PF_AHEAD) * (DOWNREC_WORDS / 4) + 6);
        }
        const uint4 a = rp[0], b = rp[1], c4 = rp[2], d = rp[3], e = rp[4], f = rp[5], g = rp[6];      // all seven requested before the test
        if (a.x == REC_NONE) continue;
#else
        const uint4 a = rp[0];
        if (a.x == REC_NONE) continue;
        const uint4 b = rp[1], c4 = rp[2], d = rp[3], e = rp[4], f = rp[5], g = rp[6];
#endif
        const uint32_t t = a.x;
        s_t[tid] = t; s_j[tid] = (uint32_t)j;
        r0 = (int)(a.y & 0xffu);
        s_rtop[tid] = (int16_t)((a.y >> 8) & 0xffu);
        nhits = (int)a.z;
        // (measured: with the sector carried in the DownRec instead of this load, the pass takes 11.3 ms instead of 10.7 ms)
        s_bsec[tid] = out.sector[t] * R;
        rowhit = out.rowhit + (int64_t)t * R;
        S.x = rs.sx[r0];
        S.y = __uint_as_float(b.x); S.z = __uint_as_float(b.y); S.s = __uint_as_float(b.z); S.t = __uint_as_float(b.w);
        S.q = __uint_as_float(c4.x); S.c00 = __uint_as_float(c4.y); S.c10 = __uint_as_float(c4.z); S.c11 = __uint_as_float(c4.w);
        S.c20 = __uint_as_float(d.x); S.c21 = __uint_as_float(d.y); S.c22 = __uint_as_float(d.z); S.c30 = __uint_as_float(d.w);
        S.c31 = __uint_as_float(e.x); S.c32 = __uint_as_float(e.y); S.c33 = __uint_as_float(e.z); S.c40 = __uint_as_float(e.w);
        S.c41 = __uint_as_float(f.x); S.c42 = __uint_as_float(f.y); S.c43 = __uint_as_float(f.z); S.c44 = __uint_as_float(f.w);
        S.chi2 = __uint_as_float(g.x);
        TC_SNAP_STORE(snap, tid, S);        // the state after the Update on r0 is the snapshot so far
        snap_row = r0; miss = 0; c_cur = -1;
        rn = rs.snd[r0];                    // >= 0: the span pass finishes seeds with nothing below r0 itself
        if (P.any_dead) for (int g = rn + 1; g < r0; ++g) rowhit[g] = -1;     // dead rows stepped over (R23) hold no hit
        phase = 2;
      }
    }
    if (__all_sync(0xffffffffu, phase == -2)) break;

    // ---- one step ----
    const bool act = phase >= 0;
    float ym = 0.0f, zm = 0.0f;
    float2 mk = make_float2(0.0f, 0.0f);
    constexpr bool SEARCH = EXT || GAP;
    const GridDesc G = desc[(SEARCH && act) ? s_bsec[tid] + rn : 0];
    if (!EXT && act && c_cur >= 0) mk = __ldg(syz + c_cur);
    SearchPre sp;
    // (A lean out-of-line search with plain loops for the gap rows was tried instead of the two span instances: fewer
    // instructions but slower, its dependent loads cost the other lanes four memory latencies where the prefetching form costs one.)
    const bool want_search = SEARCH && act && (EXT || c_cur < 0);
    const bool okp = act && kfPropagate(S, rs.sx[act ? rn : 0], P, [&](float y1, float z1, float c00, float c11) {
      if (SEARCH && want_search) searchBegin(sp, y1, z1, c00, c11, G, cell_start, P);
    });
    int32_t c = EXT ? -1 : c_cur;
    const bool known = !EXT && okp && c >= 0;
    if (SEARCH) {
      if (okp && c < 0) c = searchFinish(sp, syz, s2o, ym, zm);
    } else if (okp && c < 0) {
      cnt[CNT_ERROR] = -9;          // cannot happen: constructUp flags every seed with a gap row in its span
    }
    if (!EXT && c_cur >= 0) { ym = mk.x; zm = mk.y; }
    bool oku = false;
    if (okp && c >= 0) oku = kfUpdate(S, ym, zm, P);
    if (!act) continue;

    // ---- bookkeeping ----
    bool end_phase = !okp || (c >= 0 && !oku);       // Propagate or Update refused: the pass ends here
    const bool refused = end_phase;
    const int rb = rn;
    if (okp && !known) rowhit[rb] = oku ? c : -1;
    if (!end_phase) {
      if (oku) {
        ++nhits; snap_row = rb;
        // the search-free span instance keeps no snapshot: every step of it ends in an Update, so the live state IS the
        // snapshot; a seed whose Propagate or Update is refused there (rare) is handed to the gap instance, which redoes
        // its span from the TurnRec with snapshots (the span pass writes no row hit of a seed without gap rows)
        if (SEARCH) TC_SNAP_STORE(snap, tid, S);
        if (EXT) miss = 0;
      } else if (EXT) {
        if (++miss > P.max_row_gap) end_phase = true;
      }
    }
    bool handoff = false;
    if (!end_phase) {
      if (!EXT && rb == r0) {        // the span is done: S is the state after the Update on r0 (h0 is always known)
        if (rs.snd[rb] < 0) end_phase = true; else handoff = true;
      } else {
        rn = rs.snd[rb];
        if (rn < 0) end_phase = true;
      }
    }
    if (handoff) {
      uint4* q = down_list + (int64_t)s_j[tid] * (DOWNREC_WORDS / 4);
      q[0] = make_uint4(s_t[tid], (uint32_t)r0 | ((uint32_t)(uint16_t)s_rtop[tid] << 8), (uint32_t)nhits, 0u);
      q[1] = make_uint4(__float_as_uint(S.y), __float_as_uint(S.z), __float_as_uint(S.s), __float_as_uint(S.t));
      q[2] = make_uint4(__float_as_uint(S.q), __float_as_uint(S.c00), __float_as_uint(S.c10), __float_as_uint(S.c11));
      q[3] = make_uint4(__float_as_uint(S.c20), __float_as_uint(S.c21), __float_as_uint(S.c22), __float_as_uint(S.c30));
      q[4] = make_uint4(__float_as_uint(S.c31), __float_as_uint(S.c32), __float_as_uint(S.c33), __float_as_uint(S.c40));
      q[5] = make_uint4(__float_as_uint(S.c41), __float_as_uint(S.c42), __float_as_uint(S.c43), __float_as_uint(S.c44));
      q[6] = make_uint4(__float_as_uint(S.chi2), 0u, 0u, 0u);
      phase = -1;
    } else if (end_phase) {         // O4 step 6: output = last snapshot
      if (!SEARCH && refused) {
        gap_idx_out[atomicAdd((unsigned long long*)(cnt + CNT_N_GAP), 1ull)] = s_j[tid];
      } else {
        if (!SEARCH) TC_SNAP_STORE(snap, tid, S);     // ended on the Update of r0 with nothing below it
        writeTracklet(out, P, s_t[tid], nhits, snap_row, s_rtop[tid], snap, tid);
        if (!EXT) down_list[(int64_t)s_j[tid] * (DOWNREC_WORDS / 4)].x = REC_NONE;
      }
      phase = -1;
    } else {
      if (!EXT) {                   // pipeline: this step's hit was loaded a step ago; request the one after
        c_cur = nx_ok ? nx_raw : -1;
        const int r2 = rs.snd[rn];
        nx_ok = r2 >= r0;
        if (nx_ok) nx_raw = rowhit[r2];
      }
      const int lo = rn, hi = rb;   // dead rows stepped over (R23) hold no hit
      if (P.any_dead && hi - lo > 1)
        for (int g = lo + 1; g < hi; ++g) rowhit[g] = -1;
    }
  }
}

}  // namespace tpc
