// tpc_oracle.cpp -- plain single-threaded CPU ORACLE of the TPC sector tracker (test infrastructure).
//
// Follows DESIGN.md section 3 (formula sheet = SURVEY.md 8(c) readings R0..R27 of BASELINE.json
// north_star; PAPER.md itself gives no algorithmic detail, see tpc_oracle.h) step by step:
//   O1 grid, O2 neighbour finder, O3 cleaner + start hits, O4 tracklet constructor, O5 selector.
// No blocking, fusion or reordering.  Shares no code with the CUDA path.
//
// Build: g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC tpc_oracle.cpp -o libtpcoracle.so
// (R0: one IEEE rounding per written operation, no FMA contraction, no reassociation.)
#include "tpc_oracle.h"

#include <cmath>
#include <cstring>
#include <vector>

namespace {

inline int tri(int i, int j) { return i * (i + 1) / 2 + j; }   // i >= j, order 00,10,11,20,21,22,...

template <typename Real>
struct State {
  Real x, y, z, s, t, q;   // p = (y, z, sin(phi), dz/ds, q/pT) at plane x          (O4 "State")
  Real C[15];
  Real chi2;
};

// ---- O4 Propagate(dx): exact circle in the bend plane, series arc length; C <- F C F^T ------------
template <typename Real>
bool propagate(State<Real>& st, Real xnew, Real b, Real max_sinphi) {
  const Real dx = xnew - st.x;
  const Real s = st.s, t = st.t;
  const Real k = st.q * b;
  const Real s1 = s + dx * k;
  if (!(std::fabs(s) < max_sinphi) || !(std::fabs(s1) < max_sinphi)) return false;
  const Real one = 1;
  const Real c0 = std::sqrt(one - s * s);
  const Real c1 = std::sqrt(one - s1 * s1);
  const Real T = (s + s1) / (c0 + c1);
  const Real y1 = st.y + dx * T;
  const Real dl = dx * std::sqrt(one + T * T);
  const Real kd = k * dl;
  const Real a2 = kd * kd;
  const Real c24 = (Real)(1.0 / 24.0), c640 = (Real)(3.0 / 640.0), c6 = (Real)(1.0 / 6.0);
  const Real dS = dl * (one + a2 * c24 + a2 * a2 * c640);
  const Real z1 = st.z + t * dS;
  const Real cc = one + s * s1 + c0 * c1;
  const Real csum = c0 + c1;
  const Real c0c1 = c0 * c1;
  const Real Fys = dx * cc / (c0c1 * csum);
  const Real Fyq = dx * dx * b * cc / (c1 * csum * csum);
  const Real Fsq = dx * b;
  const Real Fzt = dS;
  const Real Fzs = t * dx * T / c0c1;
  const Real sm = (Real)0.5 * (s + s1);
  const Real cm = std::sqrt(one - sm * sm);
  const Real Fzq = t * b * dx * dx * c6 * ((Real)2 * sm / (cm * cm * cm) + s1 / (c1 * c1 * c1));
  // M = F C (full 5x5), F = I + {Fys(0,2), Fyq(0,4), Fzs(1,2), Fzt(1,3), Fzq(1,4), Fsq(2,4)}
  Real Cf[5][5], M[5][5];
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < 5; ++j) Cf[i][j] = st.C[i >= j ? tri(i, j) : tri(j, i)];
  for (int j = 0; j < 5; ++j) {
    M[0][j] = Cf[0][j] + Fys * Cf[2][j] + Fyq * Cf[4][j];
    M[1][j] = Cf[1][j] + Fzs * Cf[2][j] + Fzt * Cf[3][j] + Fzq * Cf[4][j];
    M[2][j] = Cf[2][j] + Fsq * Cf[4][j];
    M[3][j] = Cf[3][j];
    M[4][j] = Cf[4][j];
  }
  // C' = M F^T, lower triangle
  for (int i = 0; i < 5; ++i) {
    st.C[tri(i, 0)] = M[i][0] + M[i][2] * Fys + M[i][4] * Fyq;
    if (i >= 1) st.C[tri(i, 1)] = M[i][1] + M[i][2] * Fzs + M[i][3] * Fzt + M[i][4] * Fzq;
    if (i >= 2) st.C[tri(i, 2)] = M[i][2] + M[i][4] * Fsq;
    if (i >= 3) st.C[tri(i, 3)] = M[i][3];
    if (i >= 4) st.C[tri(i, 4)] = M[i][4];
  }
  st.x = xnew; st.y = y1; st.z = z1; st.s = s1;
  return true;
}

// ---- O4 Update: sequential scalar updates, y (m=0) then z (m=1); guards R12 ------------------------
template <typename Real>
bool update(State<Real>& st, Real ym, Real zm, Real err2_y, Real err2_z) {
  Real p[5] = {st.y, st.z, st.s, st.t, st.q};
  Real C[15];
  for (int i = 0; i < 15; ++i) C[i] = st.C[i];
  Real chi2 = st.chi2;
  for (int m = 0; m < 2; ++m) {
    const Real v = m == 0 ? ym : zm;
    const Real r = m == 0 ? err2_y : err2_z;
    Real Cm[5], K[5];
    for (int j = 0; j < 5; ++j) Cm[j] = C[j >= m ? tri(j, m) : tri(m, j)];
    const Real S = Cm[m] + r;
    for (int i = 0; i < 5; ++i) K[i] = Cm[i] / S;
    const Real rho = v - p[m];
    for (int i = 0; i < 5; ++i) p[i] = p[i] + K[i] * rho;
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j <= i; ++j) C[tri(i, j)] = C[tri(i, j)] - K[i] * Cm[j];
    chi2 = chi2 + rho * rho / S;
  }
  for (int i = 0; i < 5; ++i)
    if (!(C[tri(i, i)] > (Real)0)) return false;
  for (int i = 0; i < 5; ++i)
    if (!std::isfinite(p[i])) return false;
  for (int i = 0; i < 15; ++i)
    if (!std::isfinite(C[i])) return false;
  if (!std::isfinite(chi2)) return false;
  st.y = p[0]; st.z = p[1]; st.s = p[2]; st.t = p[3]; st.q = p[4];
  for (int i = 0; i < 15; ++i) st.C[i] = C[i];
  st.chi2 = chi2;
  return true;
}

// ---- O7 Rotate(alpha): the same helix seen from a frame turned by alpha about z; C <- J C J^T -------------------
template <typename Real>
bool rotate(State<Real>& st, double alpha, Real b, Real max_sinphi) {
  const Real ca = (Real)std::cos(alpha), sa = (Real)std::sin(alpha);
  const Real s = st.s, t = st.t;
  const Real c = std::sqrt((Real)1 - s * s);
  const Real s1 = s * ca - c * sa;
  if (!(std::fabs(s1) < max_sinphi)) return false;
  const Real c1 = std::sqrt((Real)1 - s1 * s1);
  const Real x1 = st.x * ca + st.y * sa;
  const Real y1 = st.y * ca - st.x * sa;
  const Real jy = c / c1, jz = -(sa * t) / c1, js = c1 / c, jq = -((st.q * b) * sa);   // jq = d s' / d y (curvature)
  Real* C = st.C;
  const Real C00 = C[0], C10 = C[1], C11 = C[2], C20 = C[3], C21 = C[4], C22 = C[5], C30 = C[6], C31 = C[7], C32 = C[8],
             C40 = C[10], C41 = C[11], C42 = C[12];
  C[0] = (jy * jy) * C00;
  C[1] = jy * (jz * C00 + C10);
  C[2] = ((jz * jz) * C00 + ((Real)2 * jz) * C10) + C11;
  const Real m2 = jq * C00 + js * C20;
  C[3] = jy * m2;
  C[4] = jz * m2 + (jq * C10 + js * C21);
  C[5] = ((jq * jq) * C00 + (((Real)2 * jq) * js) * C20) + (js * js) * C22;
  C[6] = jy * C30;
  C[7] = jz * C30 + C31;
  C[8] = jq * C30 + js * C32;
  C[10] = jy * C40;
  C[11] = jz * C40 + C41;
  C[12] = jq * C40 + js * C42;
  st.x = x1; st.y = y1; st.s = s1;
  return true;
}

// ---- O7 Match(a, b): outer state of a, rotated into b's sector if rel != 0, propagated to b's plane; diagonal chi2 ----
template <typename Real>
bool match(State<Real> a, int rel, const State<Real>& b, Real bfield, const orcParams& P, Real& chi2) {
  const double a20 = 0.3490658503988659;   // 20 degrees
  if (rel != 0 && !rotate(a, rel > 0 ? a20 : -a20, bfield, (Real)P.max_sinphi)) return false;
  if (!propagate(a, b.x, bfield, (Real)P.max_sinphi)) return false;
  const Real pa[5] = {a.y, a.z, a.s, a.t, a.q}, pb[5] = {b.y, b.z, b.s, b.t, b.q};
  Real sum = 0;
  for (int i = 0; i < 5; ++i) {
    const Real den = a.C[tri(i, i)] + b.C[tri(i, i)];
    if (!(den > (Real)0)) return false;
    const Real d = pa[i] - pb[i];
    sum = sum + (d * d) / den;
  }
  if (!(sum <= (Real)P.merge_chi2_max)) return false;
  chi2 = sum;
  return true;
}

// ---- O10 Mirror: the same helix seen from the frame turned by 180 degrees about z and walked backwards ------------
// (x, y) -> (-x, -y); the direction turns with the frame and is reversed, so sin(phi) and cos(phi) > 0 stay; z stays;
// dz/dl and the apparent charge change sign.  C <- J C J^T with J = diag(-1, +1, +1, -1, -1) over (y, z, s, t, q).
template <typename Real>
void mirror(State<Real>& st) {
  st.x = -st.x; st.y = -st.y; st.t = -st.t; st.q = -st.q;
  const int sg[5] = {-1, 1, 1, -1, -1};
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j < i; ++j)
      if (sg[i] * sg[j] < 0) st.C[tri(i, j)] = -st.C[tri(i, j)];
}

// ---- O10 LegMatch(a, b): outer states of two leg ends, b's sector d sectors after a's (d * sg >= 0) ---------------
// a is turned by alpha = d*10 + sg*90 degrees (sg = sign of a's sin phi): the frame halfway between the two sectors,
// with its x axis across the sectors in the direction a moves -- the symmetry axis of the turn, about which the two
// sides mirror each other; b is turned by -alpha and mirrored into the same frame; then as Match.
template <typename Real>
bool legMatch(State<Real> a, int d, State<Real> b, Real bfield, const orcParams& P, Real& chi2) {
  const double a10 = 0.17453292519943295, a90 = 1.5707963267948966;
  {   // R44: the two sides of a turn lie on one circle -- centres (a's frame; b's frame is turned by d * 20 degrees) close
    const Real ka = a.q * bfield, kb = b.q * bfield;
    const Real xa = a.x - a.s / ka, ya = a.y + std::sqrt((Real)1 - a.s * a.s) / ka;
    const Real xb = b.x - b.s / kb, yb = b.y + std::sqrt((Real)1 - b.s * b.s) / kb;
    const Real cd = (Real)std::cos((double)d * (2.0 * a10)), sd = (Real)std::sin((double)d * (2.0 * a10));
    const Real ex = (xb * cd - yb * sd) - xa, ey = (xb * sd + yb * cd) - ya;
    const Real md = (Real)P.leg_max_centre_dist;
    if (!(ex * ex + ey * ey <= md * md)) return false;
  }
  const double sg = a.s > (Real)0 ? 1.0 : -1.0;
  const double alpha = (double)d * a10 + sg * a90;
  if (!rotate(a, alpha, bfield, (Real)P.max_sinphi)) return false;
  if (!rotate(b, -alpha, bfield, (Real)P.max_sinphi)) return false;
  mirror(b);
  // R43: the arc of a turn is long (Propagate's arc-length series is made for row-to-row steps): eight equal steps
  const Real x0 = a.x, step = (b.x - a.x) * (Real)0.125;
  for (int i = 1; i <= 8; ++i)
    if (!propagate(a, i < 8 ? x0 + (Real)i * step : b.x, bfield, (Real)P.max_sinphi)) return false;
  const Real pa[5] = {a.y, a.z, a.s, a.t, a.q}, pb[5] = {b.y, b.z, b.s, b.t, b.q};
  Real sum = 0;
  for (int i = 0; i < 5; ++i) {
    const Real den = a.C[tri(i, i)] + b.C[tri(i, i)];
    if (!(den > (Real)0)) return false;
    const Real dd = pa[i] - pb[i];
    sum = sum + (dd * dd) / den;
  }
  if (!(sum <= (Real)P.leg_chi2_max)) return false;
  chi2 = sum;
  return true;
}

template <typename Real>
struct Tracklet {
  int status = 0;   // 0 discarded in chain fit, 1 rejected, 2 accepted
  int nhits = 0, first_row = -1, last_row = -1;
  State<Real> st{};
  std::vector<int32_t> rowhit;
};

struct Grid {   // O1, one per (sector,row) bucket
  float y0 = 0, z0 = 0, inv_e = 0;
  int ny = 0, nz = 0;
  std::vector<uint32_t> cell_start;   // [ny*nz+1], positions into sorted (bucket-local)
};

}  // namespace

struct orcResult {
  int64_t n = 0;
  int n_sectors = 0, n_rows = 0;
  bool fp64 = false, brute = false;
  std::vector<uint32_t> sorted_to_orig;
  std::vector<int32_t> cell_of_sorted, n_cells;
  std::vector<int32_t> up_raw, dn_raw, up, dn;
  std::vector<uint32_t> start_hits;
  // tracklets (stored as double regardless of Real)
  std::vector<int32_t> tl_status, tl_nhits, tl_first, tl_last, tl_rowhit;
  std::vector<double> tl_x, tl_par, tl_cov, tl_chi2;
  // tracks
  std::vector<int32_t> tr_id, tr_sector, tr_first, tr_last, tr_ncl;
  std::vector<double> tr_x, tr_par, tr_cov, tr_chi2;
  std::vector<uint32_t> tr_cl_offset, tr_cl_index;
  // O6 refit (NEXT-2): status 1 = refitted, 0 = failed; inner = state at the first kept cluster (down pass),
  // outer = state at the last kept cluster (up pass)
  std::vector<int32_t> rf_status;
  std::vector<double> rf_x_in, rf_par_in, rf_cov_in, rf_chi2, rf_x_out, rf_par_out, rf_cov_out;
  int64_t o4_ops[4] = {0, 0, 0, 0};   // Propagates, Updates, Searches, clusters inside the roads (O4)
  int64_t o2_ops[4] = {0, 0, 0, 0};   // clusters with a row pair, up candidates, down candidates, (u, d) pairs (O2)
  // O7 merger (NEXT-1)
  std::vector<int32_t> mg_next, mg_prev, mg_head;
  std::vector<double> mg_chi2;
  // O10 looper legs (rest of NEXT-1)
  std::vector<int32_t> lg_partner;
  std::vector<double> lg_chi2;
  // O12 merged tracks (NEXT-1 / NEXT-3): merged-track id and leg rank per track, cluster lists per merged track
  std::vector<int32_t> mt_id, mt_rank;
  std::vector<uint32_t> mt_cl_offset, mt_cl_index;
  // O8 cluster flags (NEXT-3)
  std::vector<uint8_t> cf_flags;
  std::vector<int32_t> cf_owner;
  std::vector<double> cf_res_y, cf_res_z;
};

namespace {

template <typename Real>
struct Tracker {
  const orcGeometry& g;
  const orcParams& P;
  const int64_t N;
  const uint32_t* off;
  const bool brute;
  const int R, S;
  std::vector<Real> Y, Z, X;           // cluster coords; row x
  std::vector<int32_t> rowOf, secOf;   // per cluster (R26: recovered from row_offset)
  std::vector<int> upRow, dnRow;       // R2
  std::vector<Grid> grids;
  std::vector<uint32_t> sorted;        // sorted_to_orig
  orcResult& res;

  Tracker(const orcGeometry& g_, const orcParams& p_, int64_t n, const uint32_t* off_, const float* y, const float* z,
          bool brute_, orcResult& r)
      : g(g_), P(p_), N(n), off(off_), brute(brute_), R(g_.n_rows), S(g_.n_sectors), res(r) {
    Y.resize(N); Z.resize(N); rowOf.resize(N); secOf.resize(N);
    for (int64_t i = 0; i < N; ++i) { Y[i] = (Real)y[i]; Z[i] = (Real)z[i]; }
    for (int s = 0; s < S; ++s)
      for (int r = 0; r < R; ++r)
        for (uint32_t i = off[s * R + r]; i < off[s * R + r + 1]; ++i) { rowOf[i] = r; secOf[i] = s; }
    X.resize(R);
    for (int r = 0; r < R; ++r) X[r] = (Real)g.row_x[r];
    // R2: up(r) = first live row among (r+1, r+2); dn(r) = first live row among (r-1, r-2)
    upRow.assign(R, -1); dnRow.assign(R, -1);
    for (int r = 0; r < R; ++r) {
      if (dead(r)) continue;
      for (int k = 1; k <= 2; ++k) if (r + k < R && !dead(r + k)) { upRow[r] = r + k; break; }
      for (int k = 1; k <= 2; ++k) if (r - k >= 0 && !dead(r - k)) { dnRow[r] = r - k; break; }
    }
  }
  bool dead(int r) const { return g.row_dead && g.row_dead[r]; }

  // ---- O1 ----------------------------------------------------------------------------------------
  int cellCoord(float v, float v0, float inv_e, int n) const {
    float f = std::floor((v - v0) * inv_e);
    if (!(f >= 0.0f)) return 0;
    if (f > (float)(n - 1)) return n - 1;
    return (int)f;
  }
  void buildGrid() {
    grids.resize((size_t)S * R);
    sorted.resize(N);
    res.cell_of_sorted.assign(N, 0);
    res.n_cells.assign((size_t)S * R, 0);
    for (int b = 0; b < S * R; ++b) {
      const int r = b % R;
      const uint32_t lo = off[b], hi = off[b + 1], n = hi - lo;
      Grid& G = grids[b];
      const float hw = g.row_x[r] * g.tan_half_sector;
      const float Wy = 2.0f * hw, Wz = g.z_max - g.z_min;
      float e = n > 0 ? std::sqrt(Wy * Wz / (float)n) : P.cell_max;
      if (e < P.cell_min) e = P.cell_min;
      if (e > P.cell_max) e = P.cell_max;
      G.y0 = -hw; G.z0 = g.z_min; G.inv_e = 1.0f / e;
      G.ny = (int)std::ceil(Wy / e); G.nz = (int)std::ceil(Wz / e);
      if (G.ny < 1) G.ny = 1;
      if (G.nz < 1) G.nz = 1;
      const int nc = G.ny * G.nz;
      res.n_cells[b] = nc;
      G.cell_start.assign(nc + 1, 0);
      std::vector<int> cell(n);
      for (uint32_t i = 0; i < n; ++i) {
        int by = cellCoord((float)Y[lo + i], G.y0, G.inv_e, G.ny);
        int bz = cellCoord((float)Z[lo + i], G.z0, G.inv_e, G.nz);
        cell[i] = bz * G.ny + by;
        G.cell_start[cell[i] + 1]++;
      }
      for (int c = 0; c < nc; ++c) G.cell_start[c + 1] += G.cell_start[c];
      std::vector<uint32_t> cur(G.cell_start.begin(), G.cell_start.end() - 1);
      for (uint32_t i = 0; i < n; ++i) {   // stable counting sort
        uint32_t pos = lo + cur[cell[i]]++;
        sorted[pos] = lo + i;
        res.cell_of_sorted[pos] = cell[i];
      }
    }
    res.sorted_to_orig = sorted;
  }

  // R3: a search is DEFINED as the predicate over all clusters of the bucket; the grid only enumerates a superset.
  template <typename F>
  void forWindow(int b, Real yc, Real zc, Real wy, Real wz, F&& f) const {
    const uint32_t lo = off[b], hi = off[b + 1];
    if (brute) {
      for (uint32_t i = lo; i < hi; ++i)
        if (std::fabs(Y[i] - yc) <= wy && std::fabs(Z[i] - zc) <= wz) f((int32_t)i);
      return;
    }
    if (hi == lo) return;
    const Grid& G = grids[b];
    // slack covers the rounding of the predicate's subtraction (superset only; predicate decides)
    const float sy = 1e-5f * ((float)std::fabs(yc) + (float)wy) + 1e-6f;
    const float sz = 1e-5f * ((float)std::fabs(zc) + (float)wz) + 1e-6f;
    const int by0 = cellCoord((float)(yc - wy) - sy, G.y0, G.inv_e, G.ny);
    const int by1 = cellCoord((float)(yc + wy) + sy, G.y0, G.inv_e, G.ny);
    const int bz0 = cellCoord((float)(zc - wz) - sz, G.z0, G.inv_e, G.nz);
    const int bz1 = cellCoord((float)(zc + wz) + sz, G.z0, G.inv_e, G.nz);
    for (int bz = bz0; bz <= bz1; ++bz)
      for (uint32_t k = G.cell_start[bz * G.ny + by0]; k < G.cell_start[bz * G.ny + by1 + 1]; ++k) {
        const uint32_t i = sorted[lo + k];
        if (std::fabs(Y[i] - yc) <= wy && std::fabs(Z[i] - zc) <= wz) f((int32_t)i);
      }
  }

  // ---- O2 ----------------------------------------------------------------------------------------
  void findNeighbours() {
    res.up_raw.assign(N, -1); res.dn_raw.assign(N, -1);
    std::vector<int32_t> U, D;
    std::vector<Real> tyu, tzu, tyd, tzd;
    for (int64_t h = 0; h < N; ++h) {
      const int r = rowOf[h], s = secOf[h];
      if (dead(r)) continue;
      const int ru = upRow[r], rd = dnRow[r];
      if (ru < 0 || rd < 0) continue;
      const Real dxu = X[ru] - X[r], dxd = X[r] - X[rd];
      const Real iu = (Real)1 / dxu, id = (Real)1 / dxd;
      const Real wyu = (Real)P.area_y * dxu, wzu = (Real)P.area_z * dxu;
      const Real wyd = (Real)P.area_y * dxd, wzd = (Real)P.area_z * dxd;
      U.clear(); D.clear(); tyu.clear(); tzu.clear(); tyd.clear(); tzd.clear();
      forWindow(s * R + ru, Y[h], Z[h], wyu, wzu, [&](int32_t u) { U.push_back(u); });
      forWindow(s * R + rd, Y[h], Z[h], wyd, wzd, [&](int32_t d) { D.push_back(d); });
      res.o2_ops[0] += 1; res.o2_ops[1] += (int64_t)U.size(); res.o2_ops[2] += (int64_t)D.size();
      res.o2_ops[3] += (int64_t)U.size() * (int64_t)D.size();          // plain counters: no arithmetic depends on them
      if (U.empty() || D.empty()) continue;
      for (int32_t u : U) { tyu.push_back((Y[u] - Y[h]) * iu); tzu.push_back((Z[u] - Z[h]) * iu); }
      for (int32_t d : D) { tyd.push_back((Y[h] - Y[d]) * id); tzd.push_back((Z[h] - Z[d]) * id); }
      bool have = false;
      Real best = 0; int32_t bu = -1, bd = -1;
      for (size_t a = 0; a < U.size(); ++a)
        for (size_t c = 0; c < D.size(); ++c) {
          const Real ey = tyu[a] - tyd[c], ez = tzu[a] - tzd[c];
          const Real dev = ey * ey + ez * ez;
          // R6: lexicographic key (Dev, orig(u), orig(d))
          bool better = !have || dev < best ||
                        (dev == best && (U[a] < bu || (U[a] == bu && D[c] < bd)));
          if (better) { have = true; best = dev; bu = U[a]; bd = D[c]; }
        }
      if (have && best <= (Real)P.link_dev2_max) { res.up_raw[h] = bu; res.dn_raw[h] = bd; }
    }
  }

  // ---- O3 ----------------------------------------------------------------------------------------
  void cleanAndStart() {
    res.up.assign(N, -1); res.dn.assign(N, -1);
    for (int64_t h = 0; h < N; ++h) {
      const int32_t u = res.up_raw[h], d = res.dn_raw[h];
      res.up[h] = (u >= 0 && res.dn_raw[u] == (int32_t)h) ? u : -1;
      res.dn[h] = (d >= 0 && res.up_raw[d] == (int32_t)h) ? d : -1;
    }
    res.start_hits.clear();
    for (int64_t h = 0; h < N; ++h)
      if (res.dn[h] == -1 && res.up[h] != -1) res.start_hits.push_back((uint32_t)h);
  }

  // ---- O4 ----------------------------------------------------------------------------------------
  // ops: how often O4 ran a Propagate, an Update, a Search, and how many clusters the Searches found inside their roads
  // (plain counters for the measurement's algorithmic operation count; no arithmetic depends on them)
  mutable int64_t ops[4] = {0, 0, 0, 0};
  int32_t search(int b, const State<Real>& st) const {
    ++ops[2];
    Real ry = (Real)P.road_sigma * std::sqrt(st.C[0] + (Real)P.err2_y);
    Real rz = (Real)P.road_sigma * std::sqrt(st.C[2] + (Real)P.err2_z);
    if (!(ry >= (Real)P.road_min)) ry = (Real)P.road_min;
    if (ry > (Real)P.road_max) ry = (Real)P.road_max;
    if (!(rz >= (Real)P.road_min)) rz = (Real)P.road_min;
    if (rz > (Real)P.road_max) rz = (Real)P.road_max;
    int32_t best = -1; Real bestd = 0;
    forWindow(b, st.y, st.z, ry, rz, [&](int32_t c) {
      ++ops[3];
      const Real dy = Y[c] - st.y, dz = Z[c] - st.z;
      const Real d2 = dy * dy + dz * dz;
      if (best < 0 || d2 < bestd || (d2 == bestd && c < best)) { best = c; bestd = d2; }
    });
    return best;
  }

  void setDiag(State<Real>& st, Real vy, Real vz) const {
    for (int i = 0; i < 15; ++i) st.C[i] = 0;
    st.C[tri(0, 0)] = vy; st.C[tri(1, 1)] = vz;
    st.C[tri(2, 2)] = (Real)P.init_var_s; st.C[tri(3, 3)] = (Real)P.init_var_t; st.C[tri(4, 4)] = (Real)P.init_var_q;
  }

  // ---- O6 refit of a selected track over its kept clusters (O6; readings R28..R30) --------
  // up pass: state from the first two kept clusters as in O4 step 1, Propagate + Update through the others in
  // ascending row -> outer state; turn (R17); down pass over all kept clusters -> inner state, chi2.
  bool refit(const uint32_t* cl, int n, State<Real>& inner, State<Real>& outer) const {
    const Real b = (Real)(0.00299792458 * (double)g.bz_tesla);
    const Real msp = (Real)P.max_sinphi, e2y = (Real)P.err2_y, e2z = (Real)P.err2_z;
    if (n < 2) return false;
    State<Real> st{};
    const uint32_t c0 = cl[0], c1 = cl[1];
    st.x = X[rowOf[c0]]; st.y = Y[c0]; st.z = Z[c0];
    {
      const Real dx = X[rowOf[c1]] - X[rowOf[c0]], dy = Y[c1] - Y[c0], dz = Z[c1] - Z[c0];
      const Real L = std::sqrt(dx * dx + dy * dy);
      st.s = dy / L; st.t = dz / L; st.q = 0;
    }
    setDiag(st, e2y, e2z);
    st.chi2 = 0;
    for (int i = 1; i < n; ++i) {
      if (!propagate(st, X[rowOf[cl[i]]], b, msp)) return false;
      if (!update(st, Y[cl[i]], Z[cl[i]], e2y, e2z)) return false;
    }
    outer = st;
    setDiag(st, (Real)P.turn_var_scale * e2y, (Real)P.turn_var_scale * e2z);
    st.chi2 = 0;
    for (int i = n - 1; i >= 0; --i) {
      if (!propagate(st, X[rowOf[cl[i]]], b, msp)) return false;
      if (!update(st, Y[cl[i]], Z[cl[i]], e2y, e2z)) return false;
    }
    inner = st;
    return true;
  }

  void refitAll() {
    const int64_t nt = (int64_t)res.tr_id.size();
    res.rf_status.assign(nt, 0);
    res.rf_x_in.assign(nt, 0); res.rf_chi2.assign(nt, 0); res.rf_x_out.assign(nt, 0);
    res.rf_par_in.assign((size_t)nt * 5, 0); res.rf_par_out.assign((size_t)nt * 5, 0);
    res.rf_cov_in.assign((size_t)nt * 15, 0); res.rf_cov_out.assign((size_t)nt * 15, 0);
    for (int64_t k = 0; k < nt; ++k) {
      const uint32_t lo = res.tr_cl_offset[k], hi = res.tr_cl_offset[k + 1];
      State<Real> in{}, out{};
      if (!refit(res.tr_cl_index.data() + lo, (int)(hi - lo), in, out)) continue;
      res.rf_status[k] = 1;
      res.rf_x_in[k] = (double)in.x; res.rf_chi2[k] = (double)in.chi2; res.rf_x_out[k] = (double)out.x;
      const Real pi[5] = {in.y, in.z, in.s, in.t, in.q}, po[5] = {out.y, out.z, out.s, out.t, out.q};
      for (int i = 0; i < 5; ++i) { res.rf_par_in[(size_t)k * 5 + i] = (double)pi[i]; res.rf_par_out[(size_t)k * 5 + i] = (double)po[i]; }
      for (int i = 0; i < 15; ++i) { res.rf_cov_in[(size_t)k * 15 + i] = (double)in.C[i]; res.rf_cov_out[(size_t)k * 15 + i] = (double)out.C[i]; }
    }
  }

  // ---- O7 links between track segments (O7; readings R31..R33) ---------------------------
  void mergeAll() {
    const int64_t nt = (int64_t)res.tr_id.size();
    res.mg_next.assign(nt, -1); res.mg_prev.assign(nt, -1); res.mg_head.assign(nt, -1); res.mg_chi2.assign(nt, 0);
    const Real bf = (Real)(0.00299792458 * (double)g.bz_tesla);
    auto stateOf = [&](int64_t k, bool outer) {
      State<Real> st{};
      const std::vector<double>& x = outer ? res.rf_x_out : res.rf_x_in;
      const std::vector<double>& p = outer ? res.rf_par_out : res.rf_par_in;
      const std::vector<double>& c = outer ? res.rf_cov_out : res.rf_cov_in;
      st.x = (Real)x[k]; st.y = (Real)p[k * 5]; st.z = (Real)p[k * 5 + 1]; st.s = (Real)p[k * 5 + 2];
      st.t = (Real)p[k * 5 + 3]; st.q = (Real)p[k * 5 + 4];
      for (int i = 0; i < 15; ++i) st.C[i] = (Real)c[k * 15 + i];
      return st;
    };
    auto relOf = [&](int sa, int sb) {          // 0 same sector, +1 / -1 azimuthal neighbour on the same side, 2 none
      if (sa == sb) return 0;
      if (S != 36 || sa / 18 != sb / 18) return 2;
      const int ja = sa % 18, jb = sb % 18;
      if (jb == (ja + 1) % 18) return 1;
      if (jb == (ja + 17) % 18) return -1;
      return 2;
    };
    std::vector<int32_t> bestB(nt, -1), bestA(nt, -1);
    std::vector<Real> chiB(nt, 0), chiA(nt, 0);
    for (int64_t a = 0; a < nt; ++a) {
      if (!res.rf_status[a]) continue;
      const State<Real> sa = stateOf(a, true);
      for (int64_t b = 0; b < nt; ++b) {
        if (b == a || !res.rf_status[b]) continue;
        const int rel = relOf(res.tr_sector[a], res.tr_sector[b]);
        if (rel == 2) continue;
        const int gap = res.tr_first[b] - res.tr_last[a];
        if (gap > P.merge_max_row_gap || gap < (rel == 0 ? 1 : -P.merge_back_rows)) continue;
        Real chi2;
        if (!match(sa, rel, stateOf(b, false), bf, P, chi2)) continue;
        if (bestB[a] < 0 || chi2 < chiB[a]) { bestB[a] = (int32_t)b; chiB[a] = chi2; }          // ties: lowest b (loop order)
        if (bestA[b] < 0 || chi2 < chiA[b]) { bestA[b] = (int32_t)a; chiA[b] = chi2; }          // ties: lowest a
      }
    }
    for (int64_t a = 0; a < nt; ++a) {
      const int32_t b = bestB[a];
      if (b >= 0 && bestA[b] == (int32_t)a) { res.mg_next[a] = b; res.mg_prev[b] = (int32_t)a; res.mg_chi2[a] = (double)chiB[a]; }
    }
    for (int64_t k = 0; k < nt; ++k) {
      int64_t h = k;
      for (int64_t guard = 0; res.mg_prev[h] >= 0 && guard < nt; ++guard) h = res.mg_prev[h];
      res.mg_head[k] = (int32_t)h;
    }
  }

  // ---- O10 looper legs: the two sides of an outer turn (O10; readings R40..R43) ------------
  void legAll() {
    const int64_t nt = (int64_t)res.tr_id.size();
    res.lg_partner.assign(nt, -1); res.lg_chi2.assign(nt, 0);
    const Real bf = (Real)(0.00299792458 * (double)g.bz_tesla);
    auto outer = [&](int64_t k) {
      State<Real> st{};
      st.x = (Real)res.rf_x_out[k]; st.y = (Real)res.rf_par_out[k * 5]; st.z = (Real)res.rf_par_out[k * 5 + 1];
      st.s = (Real)res.rf_par_out[k * 5 + 2]; st.t = (Real)res.rf_par_out[k * 5 + 3]; st.q = (Real)res.rf_par_out[k * 5 + 4];
      for (int i = 0; i < 15; ++i) st.C[i] = (Real)res.rf_cov_out[k * 15 + i];
      return st;
    };
    auto isEnd = [&](int64_t k) {                // R40: a refitted track that ends steep
      return res.rf_status[k] && !(std::fabs((Real)res.rf_par_out[k * 5 + 2]) < (Real)P.leg_min_sinphi);
    };
    auto dist = [&](int sa, int sb, int& d) {    // signed azimuthal distance a -> b on the same side
      if (sa == sb) { d = 0; return true; }
      if (S != 36 || sa / 18 != sb / 18) return false;
      d = (sb % 18 - sa % 18 + 18) % 18;
      if (d > 9) d -= 18;
      return true;
    };
    std::vector<int32_t> best(nt, -1);
    std::vector<Real> chi(nt, 0);
    for (int64_t a = 0; a < nt; ++a) {
      if (!isEnd(a)) continue;
      const State<Real> sa = outer(a);
      for (int64_t b = a + 1; b < nt; ++b) {     // R41: every pair once, the lower id is the one propagated
        if (!isEnd(b)) continue;
        int d;
        if (!dist(res.tr_sector[a], res.tr_sector[b], d) || std::abs(d) > P.leg_max_sectors) continue;
        if (std::abs(res.tr_last[a] - res.tr_last[b]) > P.leg_max_row_diff) continue;
        const State<Real> sb = outer(b);
        if (!(sa.s * sb.s < (Real)0)) continue;                  // opposite inclinations
        if ((sa.s > (Real)0 && d < 0) || (sa.s < (Real)0 && d > 0)) continue;   // a moves towards b's sector
        Real c2;
        if (!legMatch(sa, d, sb, bf, P, c2)) continue;
        if (best[a] < 0 || c2 < chi[a]) { best[a] = (int32_t)b; chi[a] = c2; }   // ties: lowest partner id (loop order:
        if (best[b] < 0 || c2 < chi[b]) { best[b] = (int32_t)a; chi[b] = c2; }   // b's partners a come in ascending a too)
      }
    }
    for (int64_t k = 0; k < nt; ++k) {            // R42: kept when reciprocal
      const int32_t o = best[k];
      if (o >= 0 && best[o] == (int32_t)k) { res.lg_partner[k] = o; res.lg_chi2[k] = (double)chi[k]; }
    }
  }

  // ---- O12 merged tracks and leg labels (O12; readings R46..R48) ------
  // A leg = an O7 chain head, next(head), ...; a merged track = one leg, or two legs whose LAST tracks are O10 partners
  // (the two sides of an outer turn).  Of two legs the primary ("first") is the one whose innermost kept
  // cluster has the smaller |z| (R48); ties -> the smaller head index.  Cluster list of a merged track: the primary leg
  // from its inner end outwards, then the secondary leg from the turn inwards -- the order along the particle's path.
  void mergedAll() {
    const int64_t nt = (int64_t)res.tr_id.size();
    res.mt_id.assign(nt, -1); res.mt_rank.assign(nt, 0);
    const bool haveLegs = (int64_t)res.lg_partner.size() == nt;
    auto tailOf = [&](int64_t k) { for (int64_t g = 0; res.mg_next[k] >= 0 && g < nt; ++g) k = res.mg_next[k]; return k; };
    auto innerAbsZ = [&](int64_t h) { return std::fabs(Z[res.tr_cl_index[res.tr_cl_offset[h]]]); };
    std::vector<int32_t> otherHead(nt, -1);
    for (int64_t h = 0; h < nt; ++h) {
      if (res.mg_head[h] != (int32_t)h) continue;          // heads only: one pass per leg
      const int64_t tl = tailOf(h);
      const int32_t p = haveLegs ? res.lg_partner[tl] : -1;
      const int32_t other = (p >= 0 && res.mg_next[p] < 0) ? res.mg_head[p] : -1;     // the partner must end its own leg
      otherHead[h] = other;
      int32_t rank = 0, id = (int32_t)h;
      if (other >= 0) {
        const Real za = innerAbsZ(h), zb = innerAbsZ(other);
        const bool primary = za < zb || (za == zb && (int32_t)h < other);
        rank = primary ? 0 : 1;
        id = (int32_t)h < other ? (int32_t)h : other;
      }
      for (int64_t k = h; k >= 0; k = res.mg_next[k]) { res.mt_id[k] = id; res.mt_rank[k] = rank; }
    }
    res.mt_cl_offset.assign(1, 0);
    res.mt_cl_index.clear();
    std::vector<int64_t> chain;
    for (int64_t k = 0; k < nt; ++k) {
      if (res.mt_id[k] == (int32_t)k && res.mg_head[k] == (int32_t)k) {   // k represents its merged track
        int64_t first = k, second = otherHead[k];
        if (second >= 0 && res.mt_rank[k] == 1) { first = second; second = k; }
        for (int64_t a = first; a >= 0; a = res.mg_next[a])
          for (uint32_t i = res.tr_cl_offset[a]; i < res.tr_cl_offset[a + 1]; ++i) res.mt_cl_index.push_back(res.tr_cl_index[i]);
        if (second >= 0) {
          chain.clear();
          for (int64_t a = second; a >= 0; a = res.mg_next[a]) chain.push_back(a);
          for (size_t c = chain.size(); c-- > 0;) {
            const int64_t a = chain[c];
            for (uint32_t i = res.tr_cl_offset[a + 1]; i-- > res.tr_cl_offset[a];) res.mt_cl_index.push_back(res.tr_cl_index[i]);
          }
        }
      }
      res.mt_cl_offset.push_back((uint32_t)res.mt_cl_index.size());
    }
  }

  // ---- O8 cluster flags (O8; readings R34..R37) ---------------------------
  void flagAll() {
    const int64_t nt = (int64_t)res.tr_id.size();
    res.cf_flags.assign(N, 0); res.cf_owner.assign(N, -1);
    res.cf_res_y.assign(N, 0); res.cf_res_z.assign(N, 0);
    const Real bf = (Real)(0.00299792458 * (double)g.bz_tesla);
    const Real msp = (Real)P.max_sinphi, tube2 = (Real)P.tube_radius * (Real)P.tube_radius;
    const bool dyn = P.tube_chi2_max > 0.0f;       // R49: the chi2 criterion of PAPER.md L108 / L114 on top of the fixed tube
    const Real sin70 = (Real)0.9396926207859084, qmax = (Real)P.inv_pt_protect;
    std::vector<Real> ownerQ(N, 0);
    std::vector<uint8_t> protAny(N, 0);          // some track that is neither low, steep nor a secondary leg has it in its tube
    const bool haveRanks = (int64_t)res.mt_rank.size() == nt;      // leg labels of O12 (else R37: every track is primary)
    for (int64_t k = 0; k < nt; ++k) {
      if (!res.rf_status[k]) continue;
      State<Real> st{};
      st.x = (Real)res.rf_x_in[k]; st.y = (Real)res.rf_par_in[k * 5]; st.z = (Real)res.rf_par_in[k * 5 + 1];
      st.s = (Real)res.rf_par_in[k * 5 + 2]; st.t = (Real)res.rf_par_in[k * 5 + 3]; st.q = (Real)res.rf_par_in[k * 5 + 4];
      for (int i = 0; i < 15; ++i) st.C[i] = (Real)res.rf_cov_in[k * 15 + i];
      const Real aq = std::fabs(st.q);
      const bool low = !(aq < qmax);
      const bool secondary = haveRanks && res.mt_rank[k] == 1;     // only the primary, first leg protects
      const int sec = res.tr_sector[k];
      const uint32_t* cl = res.tr_cl_index.data() + res.tr_cl_offset[k];
      const int ncl = (int)(res.tr_cl_offset[k + 1] - res.tr_cl_offset[k]);
      int ic = 0;
      for (int r = res.tr_first[k]; r <= res.tr_last[k]; ++r) {
        if (dead(r)) continue;
        if (r > res.tr_first[k] && !propagate(st, X[r], bf, msp)) break;
        const bool bad = low || secondary || !(std::fabs(st.s) < sin70);
        while (ic < ncl && rowOf[cl[ic]] < r) ++ic;
        const int32_t own = (ic < ncl && rowOf[cl[ic]] == r) ? (int32_t)cl[ic] : -1;     // the attached cluster of this row
        if (own >= 0) { res.cf_res_y[own] = (double)(Y[own] - st.y); res.cf_res_z[own] = (double)(Z[own] - st.z); }   // R39
        for (uint32_t c = off[sec * R + r]; c < off[sec * R + r + 1]; ++c) {
          const Real dy = Y[c] - st.y, dz = Z[c] - st.z;
          const Real d2 = dy * dy + dz * dz;
          bool in = d2 <= tube2;
          if (in && dyn) {                                  // distance in units of the track's own uncertainty on this row
            const Real x2 = (dy * dy) / (st.C[0] + (Real)P.err2_y) + (dz * dz) / (st.C[2] + (Real)P.err2_z);
            in = x2 <= (Real)P.tube_chi2_max;
          }
          if (!in && (int32_t)c != own) continue;
          if (!bad) protAny[c] = 1;                         // R36b: every good track protects what is in its tube
          if (res.cf_owner[c] < 0 || aq < ownerQ[c]) {      // ties: the lower track index (loop order)
            res.cf_owner[c] = (int32_t)k; ownerQ[c] = aq;
          }
        }
      }
    }
    for (int64_t k = 0; k < nt; ++k)
      for (uint32_t i = res.tr_cl_offset[k]; i < res.tr_cl_offset[k + 1]; ++i) res.cf_flags[res.tr_cl_index[i]] |= 1;
    for (int64_t c = 0; c < N; ++c) {
      uint8_t f = res.cf_flags[c];
      const bool has = res.cf_owner[c] >= 0, prot = has && protAny[c];
      if (has) f |= 2;
      if (prot) f |= 4;
      if (has && !prot) f |= 8;
      if (!prot) f |= 16;
      res.cf_flags[c] = f;
    }
  }

  void construct(uint32_t h0, Tracklet<Real>& T) const {
    const Real b = (Real)(0.00299792458 * (double)g.bz_tesla);
    const Real msp = (Real)P.max_sinphi, e2y = (Real)P.err2_y, e2z = (Real)P.err2_z;
    const int s = secOf[h0], r0 = rowOf[h0];
    const int32_t h1 = res.up[h0];
    const int r1 = rowOf[h1];
    T.rowhit.assign(R, -1);
    State<Real>& st = T.st;
    // 1. init from the first link
    st.x = X[r0]; st.y = Y[h0]; st.z = Z[h0];
    {
      const Real dx = X[r1] - X[r0], dy = Y[h1] - Y[h0], dz = Z[h1] - Z[h0];
      const Real L = std::sqrt(dx * dx + dy * dy);
      st.s = dy / L; st.t = dz / L; st.q = 0;
    }
    setDiag(st, e2y, e2z);
    st.chi2 = 0;
    T.rowhit[r0] = (int32_t)h0;
    int nhits = 1, rc = r0;
    // 2. chain fit
    for (int32_t h = h1; h != -1;) {
      const int r = rowOf[h];
      ++ops[0]; if (!propagate(st, X[r], b, msp)) break;
      rc = r;
      ++ops[1]; if (!update(st, Y[h], Z[h], e2y, e2z)) break;
      T.rowhit[r] = h; ++nhits;
      h = res.up[h];
    }
    if (nhits < P.min_chain_hits) { T.status = 0; T.nhits = nhits; return; }
    // 3. up-extrapolation
    int miss = 0;
    for (int r = rc + 1; r < R; ++r) {
      if (dead(r)) continue;                       // R23
      ++ops[0]; if (!propagate(st, X[r], b, msp)) break;
      const int32_t c = search(s * R + r, st);
      if (c >= 0) {
        ++ops[1]; if (!update(st, Y[c], Z[c], e2y, e2z)) break;
        T.rowhit[r] = c; ++nhits; miss = 0;
      } else if (++miss > P.max_row_gap) break;
    }
    // 4. turn (R17)
    setDiag(st, (Real)P.turn_var_scale * e2y, (Real)P.turn_var_scale * e2z);
    st.chi2 = 0;
    int rtop = -1;
    for (int r = R - 1; r >= 0; --r) if (T.rowhit[r] != -1) { rtop = r; break; }
    // 5. down pass
    int nh = 0, snap_row = -1, snap_nh = 0;
    State<Real> snap{};
    miss = 0;
    for (int r = rtop; r >= 0; --r) {
      if (dead(r)) continue;
      ++ops[0]; if (!propagate(st, X[r], b, msp)) break;
      int32_t c = T.rowhit[r];
      const bool known = c != -1;
      if (!known) c = search(s * R + r, st);
      if (c >= 0) {
        ++ops[1]; if (!update(st, Y[c], Z[c], e2y, e2z)) break;
        if (!known) T.rowhit[r] = c;
        ++nh; snap = st; snap_row = r; snap_nh = nh;
        if (r < r0) miss = 0;
      } else if (r < r0) {
        if (++miss > P.max_row_gap) break;
      }
    }
    // 6. output = last snapshot
    if (snap_row < 0) { T.status = 1; T.nhits = 0; for (auto& v : T.rowhit) v = -1; return; }
    for (int r = 0; r < snap_row; ++r) T.rowhit[r] = -1;
    T.st = snap; T.nhits = snap_nh; T.first_row = snap_row; T.last_row = rtop;
    T.status = snap_nh >= P.min_tracklet_hits ? 2 : 1;
  }

  void run() {
    if (!brute) buildGrid();
    findNeighbours();
    cleanAndStart();
    const int64_t ns = (int64_t)res.start_hits.size();
    res.tl_status.assign(ns, 0); res.tl_nhits.assign(ns, 0); res.tl_first.assign(ns, -1); res.tl_last.assign(ns, -1);
    res.tl_rowhit.assign((size_t)ns * R, -1);
    res.tl_x.assign(ns, 0); res.tl_par.assign((size_t)ns * 5, 0); res.tl_cov.assign((size_t)ns * 15, 0);
    res.tl_chi2.assign(ns, 0);
    std::vector<Real> chi2r(ns, 0);
    for (int64_t t = 0; t < ns; ++t) {
      Tracklet<Real> T;
      construct(res.start_hits[t], T);
      res.tl_status[t] = T.status; res.tl_nhits[t] = T.nhits; res.tl_first[t] = T.first_row; res.tl_last[t] = T.last_row;
      if (T.status == 0) continue;
      for (int r = 0; r < R; ++r) res.tl_rowhit[(size_t)t * R + r] = T.rowhit[r];
      res.tl_x[t] = (double)T.st.x;
      const Real p[5] = {T.st.y, T.st.z, T.st.s, T.st.t, T.st.q};
      for (int i = 0; i < 5; ++i) res.tl_par[(size_t)t * 5 + i] = (double)p[i];
      for (int i = 0; i < 15; ++i) res.tl_cov[(size_t)t * 15 + i] = (double)T.st.C[i];
      res.tl_chi2[t] = (double)T.st.chi2;
      chi2r[t] = T.st.chi2;
    }
    for (int i = 0; i < 4; ++i) res.o4_ops[i] = ops[i];
    // ---- O5 selector: owner(c) = best-priority accepted tracklet containing c -----------------------
    std::vector<int32_t> owner(N, -1);
    auto better = [&](int32_t a, int32_t bb) {   // is tracklet a of higher priority than bb ? (R19)
      if (bb < 0) return true;
      if (res.tl_nhits[a] != res.tl_nhits[bb]) return res.tl_nhits[a] > res.tl_nhits[bb];
      if (chi2r[a] != chi2r[bb]) return chi2r[a] < chi2r[bb];
      return a < bb;
    };
    for (int64_t t = 0; t < ns; ++t) {
      if (res.tl_status[t] != 2) continue;
      for (int r = 0; r < R; ++r) {
        const int32_t c = res.tl_rowhit[(size_t)t * R + r];
        if (c >= 0 && better((int32_t)t, owner[c])) owner[c] = (int32_t)t;
      }
    }
    res.tr_cl_offset.assign(1, 0);
    for (int64_t t = 0; t < ns; ++t) {
      if (res.tl_status[t] != 2) continue;
      int kept = 0, first = -1, last = -1;
      for (int r = 0; r < R; ++r) {
        const int32_t c = res.tl_rowhit[(size_t)t * R + r];
        if (c >= 0 && owner[c] == (int32_t)t) { ++kept; if (first < 0) first = r; last = r; }
      }
      if (kept < P.min_track_hits) continue;     // R20, R21: its clusters stay claimed
      for (int r = 0; r < R; ++r) {
        const int32_t c = res.tl_rowhit[(size_t)t * R + r];
        if (c >= 0 && owner[c] == (int32_t)t) res.tr_cl_index.push_back((uint32_t)c);
      }
      res.tr_cl_offset.push_back((uint32_t)res.tr_cl_index.size());
      res.tr_id.push_back((int32_t)t); res.tr_sector.push_back(secOf[res.start_hits[t]]);
      res.tr_first.push_back(first); res.tr_last.push_back(last); res.tr_ncl.push_back(kept);
      res.tr_x.push_back(res.tl_x[t]); res.tr_chi2.push_back(res.tl_chi2[t]);     // R22: not refitted
      for (int i = 0; i < 5; ++i) res.tr_par.push_back(res.tl_par[(size_t)t * 5 + i]);
      for (int i = 0; i < 15; ++i) res.tr_cov.push_back(res.tl_cov[(size_t)t * 15 + i]);
    }
  }
};

template <typename T>
void copyOut(T* dst, const std::vector<T>& v) { if (dst && !v.empty()) std::memcpy(dst, v.data(), v.size() * sizeof(T)); }

}  // namespace

extern "C" {

void orcDefaultParams(orcParams* p) {
  p->area_y = 1.5f; p->area_z = 1.5f; p->link_dev2_max = 0.64f;
  p->err2_y = 0.01f; p->err2_z = 0.01f; p->init_var_s = 1.0f; p->init_var_t = 1.0f; p->init_var_q = 100.0f;
  p->turn_var_scale = 100.0f; p->max_sinphi = 0.98f; p->road_sigma = 4.0f; p->road_min = 0.3f; p->road_max = 2.0f;
  p->max_row_gap = 4; p->min_chain_hits = 3; p->min_tracklet_hits = 10; p->min_track_hits = 10;
  p->cell_min = 0.5f; p->cell_max = 8.0f;
  p->merge_max_row_gap = 40; p->merge_back_rows = 5; p->merge_chi2_max = 50.0f;
  p->tube_radius = 1.5f; p->inv_pt_protect = 20.0f;
  p->leg_min_sinphi = 0.5f; p->leg_chi2_max = 50.0f; p->leg_max_sectors = 4; p->leg_max_row_diff = 12;
  p->leg_max_centre_dist = 10.0f;
  p->tube_chi2_max = 0.0f;
}

int orcRun(const orcGeometry* g, const orcParams* p, int64_t n, const uint32_t* off, const float* y, const float* z,
           int flags, orcResult** out) {
  if (!g || !p || !out || n < 0 || !off || g->n_sectors < 1 || g->n_rows < 3 || !g->row_x || (n > 0 && (!y || !z)))
    return ORC_ERR_INVALID_ARG;
  if (n > 0x7fffffffll) return ORC_ERR_INVALID_ARG;
  for (int r = 1; r < g->n_rows; ++r) if (!(g->row_x[r] > g->row_x[r - 1])) return ORC_ERR_INVALID_ARG;
  const int nb = g->n_sectors * g->n_rows;
  if (off[0] != 0 || (int64_t)off[nb] != n) return ORC_ERR_UNSORTED_OFFSETS;
  for (int b = 0; b < nb; ++b) if (off[b + 1] < off[b]) return ORC_ERR_UNSORTED_OFFSETS;
  for (int64_t i = 0; i < n; ++i) if (!std::isfinite(y[i]) || !std::isfinite(z[i])) return ORC_ERR_INVALID_ARG;  // R25
  orcResult* r = new orcResult();
  r->n = n; r->n_sectors = g->n_sectors; r->n_rows = g->n_rows;
  r->fp64 = (flags & ORC_FP64) != 0; r->brute = (flags & ORC_BRUTE_FORCE) != 0;
  const bool md = (flags & ORC_MERGED) != 0;
  const bool mg = md || (flags & ORC_MERGE) != 0;
  const bool fg = (flags & ORC_FLAGS) != 0;
  const bool lg = md || (flags & ORC_LEGS) != 0;
  const bool rf = mg || fg || lg || (flags & ORC_REFIT) != 0;
  if (r->fp64) { Tracker<double> T(*g, *p, n, off, y, z, r->brute, *r); T.run(); if (rf) T.refitAll(); if (mg) T.mergeAll(); if (lg) T.legAll(); if (md) T.mergedAll(); if (fg) T.flagAll(); }
  else { Tracker<float> T(*g, *p, n, off, y, z, r->brute, *r); T.run(); if (rf) T.refitAll(); if (mg) T.mergeAll(); if (lg) T.legAll(); if (md) T.mergedAll(); if (fg) T.flagAll(); }
  *out = r;
  return ORC_OK;
}
void orcFree(orcResult* r) { delete r; }

int64_t orcNumClusters(const orcResult* r) { return r->n; }
int64_t orcNumStartHits(const orcResult* r) { return (int64_t)r->start_hits.size(); }
int64_t orcNumTracks(const orcResult* r) { return (int64_t)r->tr_id.size(); }
int64_t orcNumTrackClusters(const orcResult* r) { return (int64_t)r->tr_cl_index.size(); }

void orcGetGrid(const orcResult* r, uint32_t* s2o, int32_t* cell, int32_t* ncells) {
  copyOut(s2o, r->sorted_to_orig); copyOut(cell, r->cell_of_sorted); copyOut(ncells, r->n_cells);
}
void orcGetLinks(const orcResult* r, int32_t* ur, int32_t* dr, int32_t* u, int32_t* d) {
  copyOut(ur, r->up_raw); copyOut(dr, r->dn_raw); copyOut(u, r->up); copyOut(d, r->dn);
}
void orcGetO4Counts(const orcResult* r, int64_t* four) { for (int i = 0; i < 4; ++i) four[i] = r->o4_ops[i]; }
void orcGetO2Counts(const orcResult* r, int64_t* four) { for (int i = 0; i < 4; ++i) four[i] = r->o2_ops[i]; }
void orcGetStartHits(const orcResult* r, uint32_t* sh) { copyOut(sh, r->start_hits); }
void orcGetRefit(const orcResult* r, int32_t* status, double* x_in, double* par_in, double* cov_in, double* chi2,
                 double* x_out, double* par_out, double* cov_out) {
  copyOut(status, r->rf_status); copyOut(x_in, r->rf_x_in); copyOut(par_in, r->rf_par_in); copyOut(cov_in, r->rf_cov_in);
  copyOut(chi2, r->rf_chi2); copyOut(x_out, r->rf_x_out); copyOut(par_out, r->rf_par_out); copyOut(cov_out, r->rf_cov_out);
}

void orcGetClusterFlags(const orcResult* r, uint8_t* flags, int32_t* owner) { copyOut(flags, r->cf_flags); copyOut(owner, r->cf_owner); }
void orcGetResiduals(const orcResult* r, double* ry, double* rz) { copyOut(ry, r->cf_res_y); copyOut(rz, r->cf_res_z); }
void orcGetLegs(const orcResult* r, int32_t* partner, double* chi2) { copyOut(partner, r->lg_partner); copyOut(chi2, r->lg_chi2); }
void orcGetMerged(const orcResult* r, int32_t* id, int32_t* rank, uint32_t* cl_offset, uint32_t* cl_index) {
  copyOut(id, r->mt_id); copyOut(rank, r->mt_rank); copyOut(cl_offset, r->mt_cl_offset); copyOut(cl_index, r->mt_cl_index);
}
void orcGetMerge(const orcResult* r, int32_t* next, int32_t* prev, int32_t* head, double* chi2) {
  copyOut(next, r->mg_next); copyOut(prev, r->mg_prev); copyOut(head, r->mg_head); copyOut(chi2, r->mg_chi2);
}

}  // extern "C"

namespace {
template <typename Real>
State<Real> stateFrom(const double* st, const double* cov) {
  State<Real> s{};
  s.x = (Real)st[0]; s.y = (Real)st[1]; s.z = (Real)st[2]; s.s = (Real)st[3]; s.t = (Real)st[4]; s.q = (Real)st[5];
  for (int i = 0; i < 15; ++i) s.C[i] = (Real)cov[i];
  return s;
}
template <typename Real>
int rotateT(double* st, double* cov, double alpha, double bz, double msp) {
  State<Real> s = stateFrom<Real>(st, cov);
  if (!rotate(s, alpha, (Real)(0.00299792458 * bz), (Real)msp)) return 0;
  st[0] = (double)s.x; st[1] = (double)s.y; st[2] = (double)s.z; st[3] = (double)s.s; st[4] = (double)s.t; st[5] = (double)s.q;
  for (int i = 0; i < 15; ++i) cov[i] = (double)s.C[i];
  return 1;
}
template <typename Real>
int matchT(const orcParams* p, double bz, const double* as, const double* ac, int rel, const double* bs, const double* bc,
           double* chi2) {
  Real c2 = 0;
  if (!match(stateFrom<Real>(as, ac), rel, stateFrom<Real>(bs, bc), (Real)(0.00299792458 * bz), *p, c2)) return 0;
  *chi2 = (double)c2;
  return 1;
}
template <typename Real>
void mirrorT(double* st, double* cov) {
  State<Real> s = stateFrom<Real>(st, cov);
  mirror(s);
  st[0] = (double)s.x; st[1] = (double)s.y; st[2] = (double)s.z; st[3] = (double)s.s; st[4] = (double)s.t; st[5] = (double)s.q;
  for (int i = 0; i < 15; ++i) cov[i] = (double)s.C[i];
}

template <typename Real>
int legMatchT(const orcParams* p, double bz, const double* as, const double* ac, int d, const double* bs, const double* bc,
              double* chi2) {
  Real c2;
  if (!legMatch(stateFrom<Real>(as, ac), d, stateFrom<Real>(bs, bc), (Real)(0.00299792458 * bz), *p, c2)) return 0;
  *chi2 = (double)c2;
  return 1;
}

template <typename Real>
int refitPoints(const orcGeometry* g, const orcParams* p, int n, const int32_t* rows, const double* y, const double* z,
                double* in, double* out) {
  // one sector, the given clusters (ascending rows, any number per row) as the only input
  std::vector<uint32_t> off((size_t)g->n_rows + 1, 0);
  for (int i = 0; i < n; ++i) off[rows[i] + 1]++;
  for (int r = 0; r < g->n_rows; ++r) off[r + 1] += off[r];
  std::vector<float> yf(n), zf(n);
  for (int i = 0; i < n; ++i) { yf[i] = (float)y[i]; zf[i] = (float)z[i]; }
  orcGeometry g1 = *g; g1.n_sectors = 1;
  orcResult res;
  Tracker<Real> T(g1, *p, n, off.data(), yf.data(), zf.data(), true, res);
  for (int i = 0; i < n; ++i) { T.Y[i] = (Real)y[i]; T.Z[i] = (Real)z[i]; }     // binary64 inputs stay exact
  std::vector<uint32_t> cl(n);
  for (int i = 0; i < n; ++i) cl[i] = (uint32_t)i;
  State<Real> si{}, so{};
  if (!T.refit(cl.data(), n, si, so)) return 0;
  const State<Real>* st[2] = {&si, &so};
  double* dst[2] = {in, out};
  for (int k = 0; k < 2; ++k) {     // 22 doubles: x, y, z, s, t, q, C[15], chi2
    double* d = dst[k];
    d[0] = (double)st[k]->x; d[1] = (double)st[k]->y; d[2] = (double)st[k]->z; d[3] = (double)st[k]->s;
    d[4] = (double)st[k]->t; d[5] = (double)st[k]->q;
    for (int i = 0; i < 15; ++i) d[6 + i] = (double)st[k]->C[i];
    d[21] = (double)st[k]->chi2;
  }
  return 1;
}

// One Search (O4, R13) of the clusters of one sector for the pins: the given clusters are the only input, the grid is
// built as in a run unless brute.
template <typename Real>
int searchPoints(const orcGeometry* g, const orcParams* p, int n, const int32_t* rows, const float* y, const float* z,
                 int row, const double* st, const double* cov, int brute) {
  std::vector<uint32_t> off((size_t)g->n_rows + 1, 0);
  for (int i = 0; i < n; ++i) off[rows[i] + 1]++;
  for (int r = 0; r < g->n_rows; ++r) off[r + 1] += off[r];
  orcGeometry g1 = *g; g1.n_sectors = 1;
  orcResult res;
  Tracker<Real> T(g1, *p, n, off.data(), y, z, brute != 0, res);
  if (!brute) T.buildGrid();
  return (int)T.search(row, stateFrom<Real>(st, cov));
}
}  // namespace

extern "C" {

int orcPackCharge(int64_t n, const float* q, int nb, uint16_t* code) {
  if (n < 0 || (n > 0 && (!q || !code)) || nb < 0 || nb > 14) return 0;
  for (int64_t i = 0; i < n; ++i) {
    float r = std::rint(q[i]);                       // nearest integer, ties to even
    if (!(r >= 0.0f)) r = 0.0f;                      // negative and NaN -> 0
    if (r > 65535.0f) r = 65535.0f;
    uint32_t v = (uint32_t)r;
    int L = 0;
    for (uint32_t t = v; t; t >>= 1) ++L;            // bit length
    if (L > nb + 1) {
      const int sh = L - (nb + 1);
      v = ((v + (1u << (sh - 1))) >> sh) << sh;      // to nearest, ties up; may carry into the next power of two
      const uint32_t vmax = ((1u << (nb + 1)) - 1u) << (15 - nb);
      if (v > vmax) v = vmax;
    }
    code[i] = (uint16_t)v;
  }
  return 1;
}

// O11 (rest of NEXT-4; DESIGN.md section 3 "O11", reading R45): positions -- absolute, or residuals to
// the track model -- as 16-bit integers in units of 2^-bits cm: nearest integer (ties to even), saturated; NaN -> 0.
int orcPackPositions(int64_t n, const float* y, const float* z, int bits, uint32_t* code) {
  if (n < 0 || (n > 0 && (!y || !z || !code)) || bits < 0 || bits > 15) return 0;
  const float scale = (float)(1 << bits);
  for (int64_t i = 0; i < n; ++i) {
    const float v[2] = {y[i], z[i]};
    uint32_t w = 0;
    for (int k = 0; k < 2; ++k) {
      float r = std::rint(v[k] * scale);               // a power of two: the product is exact (short of overflow)
      if (!(r == r)) r = 0.0f;
      if (r < -32768.0f) r = -32768.0f;
      if (r > 32767.0f) r = 32767.0f;
      w |= (uint32_t)(uint16_t)(int16_t)(int32_t)r << (16 * k);
    }
    code[i] = w;
  }
  return 1;
}

int orcRotate(double* state, double* cov, double alpha, double bz_tesla, double max_sinphi, int fp64) {
  return fp64 ? rotateT<double>(state, cov, alpha, bz_tesla, max_sinphi) : rotateT<float>(state, cov, alpha, bz_tesla, max_sinphi);
}
int orcMatch(const orcParams* p, double bz_tesla, const double* a_state, const double* a_cov, int rel, const double* b_state,
             const double* b_cov, int fp64, double* chi2) {
  return fp64 ? matchT<double>(p, bz_tesla, a_state, a_cov, rel, b_state, b_cov, chi2)
              : matchT<float>(p, bz_tesla, a_state, a_cov, rel, b_state, b_cov, chi2);
}

void orcMirror(double* state, double* cov) { mirrorT<double>(state, cov); }
int orcLegMatch(const orcParams* p, double bz_tesla, const double* a_state, const double* a_cov, int d, const double* b_state,
                const double* b_cov, int fp64, double* chi2) {
  return fp64 ? legMatchT<double>(p, bz_tesla, a_state, a_cov, d, b_state, b_cov, chi2)
              : legMatchT<float>(p, bz_tesla, a_state, a_cov, d, b_state, b_cov, chi2);
}

int orcRefitPoints(const orcGeometry* g, const orcParams* p, int n, const int32_t* rows, const double* y, const double* z,
                   int fp64, double* inner22, double* outer22) {
  if (!g || !p || n < 2 || !rows || !y || !z || !inner22 || !outer22) return 0;
  for (int i = 0; i < n; ++i)
    if (rows[i] < 0 || rows[i] >= g->n_rows || (i > 0 && rows[i] < rows[i - 1])) return 0;
  return fp64 ? refitPoints<double>(g, p, n, rows, y, z, inner22, outer22)
              : refitPoints<float>(g, p, n, rows, y, z, inner22, outer22);
}
void orcGetTracklets(const orcResult* r, int32_t* status, int32_t* nhits, int32_t* first, int32_t* last, int32_t* rowhit,
                     double* x, double* par, double* cov, double* chi2) {
  copyOut(status, r->tl_status); copyOut(nhits, r->tl_nhits); copyOut(first, r->tl_first); copyOut(last, r->tl_last);
  copyOut(rowhit, r->tl_rowhit); copyOut(x, r->tl_x); copyOut(par, r->tl_par); copyOut(cov, r->tl_cov);
  copyOut(chi2, r->tl_chi2);
}
void orcGetTracks(const orcResult* r, int32_t* id, int32_t* sector, int32_t* first, int32_t* last, int32_t* ncl, double* x,
                  double* par, double* cov, double* chi2, uint32_t* off, uint32_t* idx) {
  copyOut(id, r->tr_id); copyOut(sector, r->tr_sector); copyOut(first, r->tr_first); copyOut(last, r->tr_last);
  copyOut(ncl, r->tr_ncl); copyOut(x, r->tr_x); copyOut(par, r->tr_par); copyOut(cov, r->tr_cov);
  copyOut(chi2, r->tr_chi2); copyOut(off, r->tr_cl_offset); copyOut(idx, r->tr_cl_index);
}

int orcSearch(const orcGeometry* g, const orcParams* p, int n, const int32_t* rows, const float* y, const float* z, int row,
              const double* state, const double* cov, int fp64, int brute) {
  if (!g || !p || n < 0 || (n > 0 && (!rows || !y || !z)) || !state || !cov || row < 0 || row >= g->n_rows) return -2;
  for (int i = 0; i < n; ++i)
    if (rows[i] < 0 || rows[i] >= g->n_rows || (i > 0 && rows[i] < rows[i - 1])) return -2;
  return fp64 ? searchPoints<double>(g, p, n, rows, y, z, row, state, cov, brute)
              : searchPoints<float>(g, p, n, rows, y, z, row, state, cov, brute);
}

int orcPropagate(double* state, double* cov, double x_new, double bz, double max_sinphi, int fp64) {
  if (fp64) {
    State<double> st{state[0], state[1], state[2], state[3], state[4], state[5], {}, 0};
    for (int i = 0; i < 15; ++i) st.C[i] = cov[i];
    if (!propagate<double>(st, x_new, 0.00299792458 * bz, max_sinphi)) return 0;
    state[0] = st.x; state[1] = st.y; state[2] = st.z; state[3] = st.s; state[4] = st.t; state[5] = st.q;
    for (int i = 0; i < 15; ++i) cov[i] = st.C[i];
  } else {
    State<float> st{(float)state[0], (float)state[1], (float)state[2], (float)state[3], (float)state[4], (float)state[5], {}, 0};
    for (int i = 0; i < 15; ++i) st.C[i] = (float)cov[i];
    if (!propagate<float>(st, (float)x_new, (float)(0.00299792458 * (double)(float)bz), (float)max_sinphi)) return 0;
    state[0] = st.x; state[1] = st.y; state[2] = st.z; state[3] = st.s; state[4] = st.t; state[5] = st.q;
    for (int i = 0; i < 15; ++i) cov[i] = st.C[i];
  }
  return 1;
}

int orcUpdate(double* state, double* cov, double* chi2, double ym, double zm, double e2y, double e2z, int fp64) {
  if (fp64) {
    State<double> st{state[0], state[1], state[2], state[3], state[4], state[5], {}, *chi2};
    for (int i = 0; i < 15; ++i) st.C[i] = cov[i];
    if (!update<double>(st, ym, zm, e2y, e2z)) return 0;
    state[1] = st.y; state[2] = st.z; state[3] = st.s; state[4] = st.t; state[5] = st.q; *chi2 = st.chi2;
    for (int i = 0; i < 15; ++i) cov[i] = st.C[i];
  } else {
    State<float> st{(float)state[0], (float)state[1], (float)state[2], (float)state[3], (float)state[4], (float)state[5], {}, (float)*chi2};
    for (int i = 0; i < 15; ++i) st.C[i] = (float)cov[i];
    if (!update<float>(st, (float)ym, (float)zm, (float)e2y, (float)e2z)) return 0;
    state[1] = st.y; state[2] = st.z; state[3] = st.s; state[4] = st.t; state[5] = st.q; *chi2 = st.chi2;
    for (int i = 0; i < 15; ++i) cov[i] = st.C[i];
  }
  return 1;
}

}  // extern "C"
