// tpc_flags.cuh -- a8: optional per-cluster flags attached / adjacent / protected and the rejection strategies A and B
// (DESIGN.md section 3 "O8", readings R34..R37; NEXT-3 of SURVEY.md 8(f); tube of 1.5 cm, ambiguity
// to the higher-momentum track, protected = adjacent to a track with pT > 50 MeV/c and |phi| < 70 degrees).
//
// A group of FLAG_GROUP lanes per refitted track walks its rows (every lane of the group carries the same state: the
// Propagate is redundant but uniform, the candidates of a tube are shared out among the lanes).  The track walks its rows from the inner state by Propagate alone and bids for every cluster in
// its tube (found through the a1 grid: cells of the box around the tube, exact circle predicate) and for its own
// attached cluster of the row.  The bid is a 64-bit key  |q/pT| bits : track id  taken with atomicMin, so the owner is
// the track of minimal (|q/pT|, id) -- the highest momentum (R36).  Protection does not go through the owner (R36b): every
// track that is neither low-pT, nor steep on that row, nor a secondary leg (O12 rank 1, when the leg labels are given)
// sets the cluster's bit in a protection bit mask (atomicOr), so a good track protects what lies in its tube even when
// a steep or low track of higher momentum owns it.  A last pass per cluster decodes key and bit into
// the flag byte.  Keys, bits and flags are indexed by the ORIGINAL cluster index.
#pragma once
#include "tpc_kalman.cuh"
#include "tpc_select.cuh"

namespace tpc {

struct FlagIn {             // refitted tracks (device, SoA with stride cap)
  int64_t cap;
  const int32_t *status, *sector, *first_row, *last_row;
  const float *x_in, *par_in, *cov_in;
  const uint32_t *cl_offset, *cl_index;
};

// thread per track-cluster entry: the attached bit
__global__ void __launch_bounds__(256) flagAttach(const uint32_t* __restrict__ cl_index, uint8_t* __restrict__ flags,
                                                  const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= cnt[CNT_N_TRK_CL]) return;
  flags[cl_index[i]] = 1;
}

#ifndef FLAG_GROUP_
#define FLAG_GROUP_ 4
#endif
constexpr int FLAG_GROUP = FLAG_GROUP_;      // lanes per track

// CHI2 = 1: the chi2 criterion of R49 on top of the fixed tube (the walk then carries its covariance; with CHI2 = 0 the
// compiler drops the covariance transport, which no result depends on)
template <int CHI2>
__global__ void __launch_bounds__(128) flagBid(FlagIn in, const uint32_t* __restrict__ off, DevParams P, RowTables T,
                                               float tube, float chi2_max, float inv_pt_protect, const GridDesc* __restrict__ desc,
                                               const uint32_t* __restrict__ cell_start, const float2* __restrict__ syz,
                                               const uint32_t* __restrict__ s2o, unsigned long long* __restrict__ key,
                                               uint32_t* __restrict__ prot_bits, const int32_t* __restrict__ leg_rank,
                                               float2* __restrict__ walk_yz, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t k = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / FLAG_GROUP;
  const int sub = threadIdx.x % FLAG_GROUP;
  if (k >= cnt[CNT_N_TRACKS] || k >= in.cap || in.status[k] != 1) return;
  const int64_t cap = in.cap;
  const int R = P.n_rows;
  KFState S{};
  S.x = in.x_in[k];
  S.y = in.par_in[0 * cap + k]; S.z = in.par_in[1 * cap + k]; S.s = in.par_in[2 * cap + k]; S.t = in.par_in[3 * cap + k];
  S.q = in.par_in[4 * cap + k];
  S.c00 = in.cov_in[0 * cap + k]; S.c10 = in.cov_in[1 * cap + k]; S.c11 = in.cov_in[2 * cap + k]; S.c20 = in.cov_in[3 * cap + k];
  S.c21 = in.cov_in[4 * cap + k]; S.c22 = in.cov_in[5 * cap + k]; S.c30 = in.cov_in[6 * cap + k]; S.c31 = in.cov_in[7 * cap + k];
  S.c32 = in.cov_in[8 * cap + k]; S.c33 = in.cov_in[9 * cap + k]; S.c40 = in.cov_in[10 * cap + k]; S.c41 = in.cov_in[11 * cap + k];
  S.c42 = in.cov_in[12 * cap + k]; S.c43 = in.cov_in[13 * cap + k]; S.c44 = in.cov_in[14 * cap + k];
  const float aq = fabsf(S.q);
  const bool low = !(aq < inv_pt_protect) || (leg_rank != nullptr && leg_rank[k] == 1);      // or a secondary leg (L83, L86)
  const float sin70 = (float)0.9396926207859084;
  const float tube2 = tube * tube;
  const unsigned long long bid = ((unsigned long long)__float_as_uint(aq) << 32) | (unsigned long long)(uint32_t)k;
  const int sec = in.sector[k], f = in.first_row[k], l = in.last_row[k];
  const int bsec = sec * R;
  const uint32_t* cl = in.cl_index + in.cl_offset[k];
  const int ncl = (int)(in.cl_offset[k + 1] - in.cl_offset[k]);
  int ic = 0;
  for (int r = f; r <= l; ++r) {
    if (T.dead[r]) continue;
    if (r > f && !kfPropagate(S, T.row_x[r], P, [](float, float, float, float) {})) break;
    const bool good = !low && fabsf(S.s) < sin70;
    // the attached cluster of this row (R35): the list is in ascending row, rows follow from row_offset (R26)
    const uint32_t b_lo = __ldg(off + bsec + r), b_hi = __ldg(off + bsec + r + 1);
    while (ic < ncl && cl[ic] < b_lo) ++ic;
    if (sub == 0 && ic < ncl && cl[ic] < b_hi) {
      const uint32_t own = cl[ic];
      atomicMin(key + own, bid);
      if (good) atomicOr(prot_bits + (own >> 5), 1u << (own & 31u));
      // for the track-model residuals (R39): the walking state at the attached cluster, in the order of the track's
      // cluster list (consecutive writes); flagResiduals turns them into residuals in one pass over all lists
      if (walk_yz) walk_yz[in.cl_offset[k] + ic] = make_float2(S.y, S.z);
    }
    // the tube: cells of the box around it (a hair wider than the tube: fl(dy*dy) <= fl(tube*tube) does not quite imply
    // |dy| <= tube), exact circle predicate; the lanes of the group take the candidates of a cell row in turn
    const GridDesc G = desc[bsec + r];
    if (G.n == 0) continue;
    const float yc = S.y, zc = S.z, w = tube * 1.000001f;
    const float sy = 1e-5f * (fabsf(yc) + w) + 1e-6f, sz = 1e-5f * (fabsf(zc) + w) + 1e-6f;     // superset slack (R3)
    const int by0 = cellCoord((yc - w) - sy, G.y0, G.inv_e, G.ny), by1 = cellCoord((yc + w) + sy, G.y0, G.inv_e, G.ny);
    const int bz0 = cellCoord((zc - w) - sz, G.z0, G.inv_e, G.nz), bz1 = cellCoord((zc + w) + sz, G.z0, G.inv_e, G.nz);
    const uint32_t* cs = cell_start + G.cell_base + by0;
    for (int bz = bz0; bz <= bz1; ++bz) {
      const uint32_t k0 = __ldg(cs + bz * G.ny), k1 = __ldg(cs + bz * G.ny + (by1 - by0 + 1));
      for (uint32_t i = k0 + sub; i < k1; i += FLAG_GROUP) {
        const float2 c = __ldg(syz + i);
        const float dy = c.x - yc, dz = c.y - zc;
        const float d2 = dy * dy + dz * dz;
        bool inside = d2 <= tube2;
        if (CHI2 && inside) {
          const float x2 = (dy * dy) / (S.c00 + P.err2_y) + (dz * dz) / (S.c11 + P.err2_z);
          inside = x2 <= chi2_max;
        }
        if (inside) {
          const uint32_t o = __ldg(s2o + i);
          atomicMin(key + o, bid);
          if (good) atomicOr(prot_bits + (o >> 5), 1u << (o & 31u));
        }
      }
    }
  }
}

// O11 (rest of NEXT-4; DESIGN.md section 3 "O11", reading R45): a position or residual in units of
// 2^-pos_bits cm as a 16-bit integer: nearest (ties to even), saturated, NaN -> 0; two per word, y16 | z16 << 16
__device__ __forceinline__ uint32_t posCode16(float v, float scale) {
  float r = rintf(v * scale);
  if (!(r == r)) r = 0.0f;
  r = fminf(fmaxf(r, -32768.0f), 32767.0f);
  return (uint32_t)(uint16_t)(int16_t)(int32_t)r;
}
__device__ __forceinline__ uint32_t posCode(float y, float z, float scale) { return posCode16(y, scale) | (posCode16(z, scale) << 16); }

// thread per track-cluster entry: res = cluster - walking state of its track on its row (R39); entries the walk did not
// reach (refused Propagate, track not refitted) still hold the NaN pattern the buffer was filled with
__global__ void __launch_bounds__(256) flagResiduals(const uint32_t* __restrict__ cl_index, const float2* __restrict__ walk_yz,
                                                     const float* __restrict__ yin, const float* __restrict__ zin,
                                                     float* __restrict__ res_y, float* __restrict__ res_z,
                                                     uint32_t* __restrict__ res_code, int pos_bits,
                                                     const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= cnt[CNT_N_TRK_CL]) return;
  const float2 w = walk_yz[i];
  if (!(w.x == w.x)) return;
  const uint32_t c = cl_index[i];
  const float ry = yin[c] - w.x, rz = zin[c] - w.y;
  if (res_y) { res_y[c] = ry; res_z[c] = rz; }
  if (res_code) res_code[c] = posCode(ry, rz, (float)(1 << pos_bits));       // O11
}

// thread per cluster: key -> flag byte and owner
__global__ void __launch_bounds__(256) flagFinish(int64_t N, const unsigned long long* __restrict__ key,
                                                  const uint32_t* __restrict__ prot_bits, uint8_t* __restrict__ flags,
                                                  int32_t* __restrict__ owner, const int64_t* __restrict__ cnt) {
  if (cnt[CNT_ERROR] != 0) return;
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= N) return;
  const unsigned long long kk = key[c];
  const bool has = kk != ~0ull;
  const bool prot = has && ((prot_bits[c >> 5] >> (c & 31)) & 1u) != 0u;
  uint8_t fl = flags[c] & 1;
  if (has) fl |= 2;
  if (prot) fl |= 4;
  if (has && !prot) fl |= 8;
  if (!prot) fl |= 16;
  flags[c] = fl;
  owner[c] = has ? (int32_t)(kk & 0x7fffffffull) : -1;
}

// a9 (part of NEXT-4; DESIGN.md section 3 "O9"): dynamic-precision 16-bit code of the cluster charges.
// Streaming: 4 bytes in, 2 bytes out per cluster; eight clusters per thread (two 16-byte loads, one 16-byte store).
__device__ __forceinline__ uint32_t packOne(float q, int nb) {
  float r = rintf(q);                              // nearest integer, ties to even
  if (!(r >= 0.0f)) r = 0.0f;                      // negative and NaN -> 0
  if (r > 65535.0f) r = 65535.0f;
  uint32_t v = (uint32_t)r;
  const int L = 32 - __clz(v);                     // bit length (0 for v = 0)
  if (L > nb + 1) {
    const int sh = L - (nb + 1);
    v = ((v + (1u << (sh - 1))) >> sh) << sh;      // to nearest, ties up
    v = min(v, ((1u << (nb + 1)) - 1u) << (15 - nb));
  }
  return v;
}

__global__ void __launch_bounds__(256) packCharge(int64_t N, const float* __restrict__ q, int nb, uint16_t* __restrict__ code) {
  const int64_t i8 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 8;
  if (i8 >= N) return;
  if (i8 + 8 <= N && (((uintptr_t)q | (uintptr_t)code) & 15) == 0) {     // eight clusters: 2 x 16 bytes in, 16 bytes out
    const float4 v = __ldcs(reinterpret_cast<const float4*>(q + i8));
    const float4 w = __ldcs(reinterpret_cast<const float4*>(q + i8) + 1);
    uint4 o;
    o.x = packOne(v.x, nb) | (packOne(v.y, nb) << 16); o.y = packOne(v.z, nb) | (packOne(v.w, nb) << 16);
    o.z = packOne(w.x, nb) | (packOne(w.y, nb) << 16); o.w = packOne(w.z, nb) | (packOne(w.w, nb) << 16);
    __stcs(reinterpret_cast<uint4*>(code + i8), o);
  } else {
    for (int64_t i = i8; i < min(i8 + 8, N); ++i) code[i] = (uint16_t)packOne(q[i], nb);
  }
}

// O11 of the absolute positions.  Streaming: 8 bytes in, 4 bytes out per cluster; four clusters per thread.
__global__ void __launch_bounds__(256) packPositions(int64_t N, const float* __restrict__ y, const float* __restrict__ z,
                                                     int pos_bits, uint32_t* __restrict__ code) {
  const int64_t i4 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (i4 >= N) return;
  const float scale = (float)(1 << pos_bits);
  if (i4 + 4 <= N && (((uintptr_t)y | (uintptr_t)z | (uintptr_t)code) & 15) == 0) {
    const float4 a = __ldcs(reinterpret_cast<const float4*>(y + i4));
    const float4 b = __ldcs(reinterpret_cast<const float4*>(z + i4));
    __stcs(reinterpret_cast<uint4*>(code + i4),
           make_uint4(posCode(a.x, b.x, scale), posCode(a.y, b.y, scale), posCode(a.z, b.z, scale), posCode(a.w, b.w, scale)));
  } else {
    for (int64_t i = i4; i < min(i4 + 4, N); ++i) code[i] = posCode(y[i], z[i], scale);
  }
}

}  // namespace tpc
