// tpc_merged.cuh -- a11: optional merged tracks and leg labels (DESIGN.md section 3 "O12", readings R46..R48; rest of
// NEXT-1 and what NEXT-3 needs of it; "only the primary, first leg is protected", L86, L92 "merging of track
// segments and legs of the same track").
//
// A leg = a chain of the a7 merger (head, next(head), ...); a merged track = one leg, or two legs whose LAST tracks are
// partners of the a10 leg pairing (the two sides of an outer turn).  Of two legs the primary one is that whose innermost
// kept cluster has the smaller |z| (R48; ties: the smaller head index).  Per track: the merged track it belongs to (named
// by the smaller head index) and the rank of its leg (0 primary, 1 secondary); per merged track, at the index of the
// track that names it: its clusters in the order along the particle's path -- the primary leg from its inner end outwards,
// then the secondary leg from the turn inwards.  Chains are a handful of segments long: every track walks its own.
#pragma once
#include "tpc_common.cuh"

namespace tpc {

struct MergedIn {
  int64_t cap;
  const int32_t *next, *head, *partner;       // a7, a10
  const uint32_t *cl_offset, *cl_index;       // a5: kept clusters per track, original indices, ascending row
  const float* z;                             // input z by original index
};
struct MergedOut {
  int32_t *id, *rank;        // [cap_tracks]
  uint32_t* cl_offset;       // [cap_tracks + 1]: first the lengths, then (scanned in place) the offsets
  uint32_t* cl_index;        // [cap_track_clusters]
};

// thread per track: id and rank of its leg; the naming track also counts the clusters of the merged track
__global__ void __launch_bounds__(256) mergedLabel(MergedIn in, MergedOut out, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nt = min(cnt[CNT_N_TRACKS], in.cap);
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k > nt) return;
  if (k == nt) { out.cl_offset[k] = 0u; return; }        // the closing entry of the scan
  const int32_t h = in.head[k];
  int64_t tl = k;
  for (int64_t g = 0; g < nt; ++g) { const int32_t n = in.next[tl]; if (n < 0) break; tl = n; }
  const int32_t p = in.partner[tl];
  const int32_t other = (p >= 0 && in.next[p] < 0) ? in.head[p] : -1;       // the partner must end its own leg
  int32_t id = h, rank = 0;
  if (other >= 0) {
    const float za = fabsf(in.z[in.cl_index[in.cl_offset[h]]]), zb = fabsf(in.z[in.cl_index[in.cl_offset[other]]]);
    const bool primary = za < zb || (za == zb && h < other);
    rank = primary ? 0 : 1;
    id = min(h, other);
  }
  out.id[k] = id; out.rank[k] = rank;
  uint32_t len = 0;
  if (id == (int32_t)k && h == (int32_t)k) {
    for (int32_t a = h; a >= 0; a = in.next[a]) len += in.cl_offset[a + 1] - in.cl_offset[a];
    for (int32_t a = other; a >= 0; a = in.next[a]) len += in.cl_offset[a + 1] - in.cl_offset[a];
  }
  out.cl_offset[k] = len;
}

// thread per naming track: copy the cluster lists of its one or two legs in path order
__global__ void __launch_bounds__(128) mergedFill(MergedIn in, MergedOut out, int64_t cap_cl, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t nt = min(cnt[CNT_N_TRACKS], in.cap);
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nt || out.id[k] != (int32_t)k || in.head[k] != (int32_t)k) return;
  uint32_t w = out.cl_offset[k];
  const uint32_t end = out.cl_offset[k + 1];
  if ((int64_t)end > cap_cl) return;                      // capacity overflow is reported by the selector already
  int32_t tl = (int32_t)k;
  for (int64_t g = 0; g < nt; ++g) { const int32_t n = in.next[tl]; if (n < 0) break; tl = n; }
  const int32_t p = in.partner[tl];
  const int32_t other = (p >= 0 && in.next[p] < 0) ? in.head[p] : -1;
  int32_t first = (int32_t)k, second = other;
  if (other >= 0 && out.rank[k] == 1) { first = other; second = (int32_t)k; }
  for (int32_t a = first; a >= 0; a = in.next[a])
    for (uint32_t i = in.cl_offset[a]; i < in.cl_offset[a + 1]; ++i) out.cl_index[w++] = in.cl_index[i];
  if (second >= 0) {
    // the secondary leg backwards: from its last segment to its head, every segment from its last cluster to its first.
    // Chains are short: the walk to the segment in front of `stop` is repeated per segment instead of storing the chain.
    int32_t stop = -1;                                     // the segment written last
    for (;;) {
      int32_t a = second;
      while (in.next[a] != stop) a = in.next[a];
      for (uint32_t i = in.cl_offset[a + 1]; i-- > in.cl_offset[a];) out.cl_index[w++] = in.cl_index[i];
      if (a == second) break;
      stop = a;
    }
  }
}

}  // namespace tpc
