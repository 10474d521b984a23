// tpcgen.cpp -- seeded synthetic TPC cluster generator (input recipe: DESIGN.md "Input recipe";
// SURVEY.md section 8(d); BASELINE.json configs 0-4).
//
// This module serves BOTH the oracle tests and the CUDA path with inputs.  It holds none of the
// tracker's arithmetic (no grid, no links, no Kalman filter): it only draws helices from a vertex,
// intersects them analytically with the pad-row planes of each sector, smears and shuffles.
// It stands in for the ALICE pp / simulated Pb-Pb data of the paper (Fig. 4, L106 Fig. 6),
// which are not available.
//
// All math in fp64, results rounded once to fp32.  The random numbers come from a counter-based
// generator (SplitMix64 finaliser over (seed, stream, index, counter)), so the data do not depend on
// thread count or generation order.
//
// Build: g++ -O2 -shared -fPIC -fopenmp tpcgen.cpp -o libtpcgen.so
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

extern "C" {

typedef struct {
  int32_t kind;        // 0: pT log-uniform on [pt_lo,pt_hi]; 1: pT ~ pT*exp(-pT/pt_scale) truncated to
                       // [pt_lo,pt_hi]; 2: pT uniform on [pt_lo,pt_hi]
  int32_t max_turns;   // helix turns followed (1 for primaries that leave, 2 for loopers)
  int64_t n_tracks;    // tracks of this population (per event; ignored for pile-up collisions)
  double pt_lo, pt_hi, pt_scale;
  double phi_lo, phi_hi;   // global azimuth of the initial direction, radians
  double eta_max;          // eta uniform in [-eta_max, eta_max]
} tpcgenPopulation;

typedef struct {
  uint64_t seed;
  int32_t n_sectors;       // 1 (single sector, both z signs kept in it) or 36 (18 azimuthal x 2 sides)
  int32_t n_rows;
  const double* row_x;     // [n_rows] local x of the pad-row planes, cm
  double bz_tesla;
  double tan_half_sector;  // tan(10 deg)
  double z_abs_max;        // 250 cm: drift length; crossings with |z_true| above are dropped
  double sigma_y, sigma_z; // Gaussian smearing, cm
  double noise_frac;       // noise clusters = noise_frac * (track clusters), uniform in (sector,row,y,z)
  double vtx_sigma_z;      // vertex z ~ N(0, vtx_sigma_z)
  int32_t n_collisions;    // <=1: one event made of pop[0..n_pop); >1: pile-up time frame, every
                           // collision draws its multiplicity (below) from pop[0]'s spectrum
  int32_t n_pop;
  const tpcgenPopulation* pop;
  double mult_mean, mult_cap;  // per-collision track count ~ Exp(mean) truncated (rejection) at cap
  double t0_window_us;         // interaction time uniform in [0, window]
  double v_drift_cm_per_us;    // z shift = v_drift * t0 toward / through the central plane
} tpcgenConfig;

struct tpcgenData {
  int32_t n_sectors = 0, n_rows = 0;
  std::vector<uint32_t> row_offset;          // [n_sectors*n_rows+1]
  std::vector<float> x, y, z, q;             // [n_clusters]
  std::vector<int32_t> truth_track;          // [n_clusters] generating track id, -1 = noise
  std::vector<int32_t> truth_turn;           // [n_clusters] helix turn number (0 = first), -1 noise
  // per-track truth, [n_tracks]
  std::vector<double> t_pt, t_phi0, t_eta, t_vz, t_zshift;
  std::vector<int32_t> t_charge_sign;        // h = +1/-1: direction angle = phi0 - h*psi
};

}  // extern "C"

namespace {

inline uint64_t mix64(uint64_t v) {
  v += 0x9E3779B97F4A7C15ull;
  v = (v ^ (v >> 30)) * 0xBF58476D1CE4E5B9ull;
  v = (v ^ (v >> 27)) * 0x94D049BB133111EBull;
  return v ^ (v >> 31);
}
// counter-based: value depends only on (seed, stream, index, counter)
inline uint64_t rnd_u64(uint64_t seed, uint64_t stream, uint64_t index, uint64_t counter) {
  uint64_t h = mix64(seed ^ 0xA0761D6478BD642Full);
  h = mix64(h ^ (stream * 0xE7037ED1A0B428DBull));
  h = mix64(h ^ (index * 0x8EBC6AF09C88C6E3ull));
  h = mix64(h ^ (counter * 0x589965CC75374CC3ull));
  return h;
}
inline double rnd_uniform(uint64_t seed, uint64_t stream, uint64_t index, uint64_t counter) {
  return ((rnd_u64(seed, stream, index, counter) >> 11) + 0.5) * (1.0 / 9007199254740992.0);  // (0,1)
}
inline double rnd_normal(uint64_t seed, uint64_t stream, uint64_t index, uint64_t counter) {
  // Box-Muller on two counters (2*counter, 2*counter+1)
  double u1 = rnd_uniform(seed, stream, index, 2 * counter);
  double u2 = rnd_uniform(seed, stream, index, 2 * counter + 1);
  return std::sqrt(-2.0 * std::log(u1)) * std::cos(6.283185307179586476925 * u2);
}

enum : uint64_t { ST_TRACK = 1, ST_SMEAR = 2, ST_NOISE = 3, ST_SHUFFLE = 4, ST_COLL = 5 };

struct RawCluster {
  int32_t bucket;  // sector*n_rows + row
  float y, z;
  int32_t track, turn;
  uint64_t key;    // shuffle key
};

double draw_pt(const tpcgenPopulation& p, uint64_t seed, uint64_t tid) {
  if (p.kind == 0) {
    double u = rnd_uniform(seed, ST_TRACK, tid, 0);
    return p.pt_lo * std::exp(u * std::log(p.pt_hi / p.pt_lo));
  } else if (p.kind == 2) {
    double u = rnd_uniform(seed, ST_TRACK, tid, 0);
    return p.pt_lo + u * (p.pt_hi - p.pt_lo);
  }
  // Gamma(shape 2, scale) = sum of two exponentials; truncate by rejection
  for (uint64_t att = 0;; ++att) {
    double u1 = rnd_uniform(seed, ST_TRACK, tid, 100 + 2 * att);
    double u2 = rnd_uniform(seed, ST_TRACK, tid, 101 + 2 * att);
    double pt = -p.pt_scale * (std::log(u1) + std::log(u2));
    if (pt >= p.pt_lo && pt <= p.pt_hi) return pt;
  }
}

}  // namespace

extern "C" {

tpcgenData* tpcgen_generate(const tpcgenConfig* c) {
  if (!c || !c->row_x || c->n_rows <= 0 || (c->n_sectors != 1 && c->n_sectors != 36) || c->n_pop <= 0 || !c->pop)
    return nullptr;
  const double kPi = 3.14159265358979323846;
  const double kTwoPi = 2.0 * kPi;
  const int n_az = (c->n_sectors == 1) ? 1 : 18;
  const bool split_sides = (c->n_sectors == 36);
  const double radius_per_pt = 1.0 / (0.00299792458 * std::fabs(c->bz_tesla));  // cm per GeV/c
  const double bsign = c->bz_tesla >= 0 ? 1.0 : -1.0;
  const int R = c->n_rows;
  const double r_in = c->row_x[0];
  const double r_out = c->row_x[R - 1] * std::sqrt(1.0 + c->tan_half_sector * c->tan_half_sector);

  tpcgenData* d = new tpcgenData();
  d->n_sectors = c->n_sectors;
  d->n_rows = R;

  // ---- 1. track list -------------------------------------------------------------------------
  struct Trk { int pop; double zshift; double vz; };
  std::vector<Trk> trks;
  if (c->n_collisions <= 1) {
    double vz = c->vtx_sigma_z > 0 ? c->vtx_sigma_z * rnd_normal(c->seed, ST_COLL, 0, 0) : 0.0;
    for (int p = 0; p < c->n_pop; ++p)
      for (int64_t i = 0; i < c->pop[p].n_tracks; ++i) trks.push_back({p, 0.0, vz});
  } else {
    for (int k = 0; k < c->n_collisions; ++k) {
      int64_t mult = 0;
      for (uint64_t att = 0;; ++att) {
        double u = rnd_uniform(c->seed, ST_COLL, k, 10 + att);
        double m = -c->mult_mean * std::log(1.0 - u);
        if (m <= c->mult_cap) { mult = (int64_t)m; break; }
      }
      double t0 = c->t0_window_us * rnd_uniform(c->seed, ST_COLL, k, 1);
      double vz = c->vtx_sigma_z > 0 ? c->vtx_sigma_z * rnd_normal(c->seed, ST_COLL, k, 1) : 0.0;
      for (int64_t i = 0; i < mult; ++i) trks.push_back({0, c->v_drift_cm_per_us * t0, vz});
    }
  }
  const int64_t nt = (int64_t)trks.size();
  d->t_pt.resize(nt); d->t_phi0.resize(nt); d->t_eta.resize(nt); d->t_vz.resize(nt);
  d->t_zshift.resize(nt); d->t_charge_sign.resize(nt);

  // ---- 2. crossings --------------------------------------------------------------------------
  const int64_t kChunk = 512;
  const int64_t n_chunks = (nt + kChunk - 1) / kChunk;
  std::vector<std::vector<RawCluster>> chunk_out((size_t)n_chunks);
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t ch = 0; ch < n_chunks; ++ch) {
    std::vector<RawCluster>& out = chunk_out[(size_t)ch];
    const int64_t t_end = std::min(nt, (ch + 1) * kChunk);
    for (int64_t t = ch * kChunk; t < t_end; ++t) {
      const tpcgenPopulation& P = c->pop[trks[t].pop];
      const double pt = draw_pt(P, c->seed, (uint64_t)t);
      const double phi0 = P.phi_lo + (P.phi_hi - P.phi_lo) * rnd_uniform(c->seed, ST_TRACK, t, 1);
      const double eta = P.eta_max * (2.0 * rnd_uniform(c->seed, ST_TRACK, t, 2) - 1.0);
      const double chg = rnd_uniform(c->seed, ST_TRACK, t, 3) < 0.5 ? -1.0 : 1.0;
      const double h = chg * bsign;   // direction angle = phi0 - h*psi
      const double Rh = pt * radius_per_pt;
      const double tanl = std::sinh(eta);
      d->t_pt[t] = pt; d->t_phi0[t] = phi0; d->t_eta[t] = eta; d->t_vz[t] = trks[t].vz;
      d->t_zshift[t] = trks[t].zshift; d->t_charge_sign[t] = (int32_t)h;
      if (2.0 * Rh <= r_in) continue;   // never reaches the first pad row
      // azimuth intervals swept while the distance from the beam line is inside [r_in, r_out]:
      // point at turning angle psi has distance 2R sin(psi/2) and azimuth phi0 - h*psi/2.
      const double a1 = std::asin(r_in / (2.0 * Rh));
      const double a2 = (r_out >= 2.0 * Rh) ? 0.5 * kPi : std::asin(r_out / (2.0 * Rh));
      bool cand[18];
      for (int a = 0; a < n_az; ++a) {
        const double alpha = (a + 0.5) * (kTwoPi / 18.0);
        // is alpha within (half-sector + margin) of phi0 - h*[a1,a2] or phi0 - h*[pi-a2, pi-a1] ?
        auto near = [&](double lo, double hi) {
          double c0 = phi0 - h * 0.5 * (lo + hi), hw = 0.5 * (hi - lo) + 0.20;  // 0.20 rad > 10 deg
          double dlt = std::remainder(alpha - c0, kTwoPi);
          return std::fabs(dlt) <= hw;
        };
        cand[a] = near(a1, a2) || near(kPi - a2, kPi - a1);
      }
      for (int a = 0; a < n_az; ++a) {
        if (!cand[a]) continue;
        const double alpha = (a + 0.5) * (kTwoPi / 18.0);
        const double delta = phi0 - alpha;
        const double sd = std::sin(delta), cd = std::cos(delta);
        for (int r = 0; r < R; ++r) {
          const double xr = c->row_x[r];
          const double v = sd - h * xr / Rh;      // sin(theta) at the crossing, theta = delta - h*psi
          if (!(std::fabs(v) < 1.0)) continue;
          const double as = std::asin(v);
          for (int sol = 0; sol < 2; ++sol) {
            const double theta = sol == 0 ? as : kPi - as;
            double psi = h * (delta - theta);
            psi -= kTwoPi * std::floor(psi / kTwoPi);   // [0, 2pi)
            const double yl = -h * Rh * (cd - std::cos(theta));
            if (std::fabs(yl) > xr * c->tan_half_sector) continue;
            for (int k = 0; k < P.max_turns; ++k) {
              const double zt = trks[t].vz + Rh * (psi + kTwoPi * k) * tanl;
              if (std::fabs(zt) > c->z_abs_max) break;
              int side = (split_sides && zt < 0) ? 1 : 0;
              double zs = zt;
              if (trks[t].zshift != 0.0) zs = (zt >= 0) ? zt - trks[t].zshift : zt + trks[t].zshift;
              const uint64_t cid = ((uint64_t)a * R + r) * 2 * 8 + (uint64_t)sol * 8 + k;   // k < 8
              const double ys = yl + c->sigma_y * rnd_normal(c->seed, ST_SMEAR, (uint64_t)t, 2 * cid);
              const double zz = zs + c->sigma_z * rnd_normal(c->seed, ST_SMEAR, (uint64_t)t, 2 * cid + 1);
              RawCluster rc;
              rc.bucket = (a + 18 * side) * R + r;
              rc.y = (float)ys; rc.z = (float)zz; rc.track = (int32_t)t; rc.turn = k;
              rc.key = rnd_u64(c->seed, ST_SHUFFLE, (uint64_t)t, cid);
              out.push_back(rc);
            }
          }
        }
      }
    }
  }
  std::vector<RawCluster> all;
  {
    size_t tot = 0;
    for (auto& v : chunk_out) tot += v.size();
    all.reserve(tot + (size_t)(c->noise_frac * (double)tot) + 16);
    for (auto& v : chunk_out) { all.insert(all.end(), v.begin(), v.end()); std::vector<RawCluster>().swap(v); }
  }
  // ---- 3. noise ------------------------------------------------------------------------------
  const int64_t n_trk_cl = (int64_t)all.size();
  const int64_t n_noise = (int64_t)std::floor(c->noise_frac * (double)n_trk_cl);
  const bool frame = c->n_collisions > 1;
  for (int64_t i = 0; i < n_noise; ++i) {
    int s = (int)(rnd_uniform(c->seed, ST_NOISE, i, 0) * c->n_sectors);
    int r = (int)(rnd_uniform(c->seed, ST_NOISE, i, 1) * R);
    if (s >= c->n_sectors) s = c->n_sectors - 1;
    if (r >= R) r = R - 1;
    double hw = c->row_x[r] * c->tan_half_sector;
    double y = hw * (2.0 * rnd_uniform(c->seed, ST_NOISE, i, 2) - 1.0);
    double u = rnd_uniform(c->seed, ST_NOISE, i, 3);
    double z;
    if (frame || !split_sides) z = c->z_abs_max * (2.0 * u - 1.0);
    else z = (s < 18) ? c->z_abs_max * u : -c->z_abs_max * u;
    RawCluster rc;
    rc.bucket = s * R + r; rc.y = (float)y; rc.z = (float)z; rc.track = -1; rc.turn = -1;
    rc.key = rnd_u64(c->seed, ST_SHUFFLE, 0xFFFFFFFFFFull + (uint64_t)i, 0);
    all.push_back(rc);
  }
  // ---- 4. bucket by (sector,row) and shuffle inside each bucket --------------------------------
  const int64_t N = (int64_t)all.size();
  const int nb = c->n_sectors * R;
  d->row_offset.assign(nb + 1, 0);
  for (const RawCluster& rc : all) d->row_offset[rc.bucket + 1]++;
  for (int b = 0; b < nb; ++b) d->row_offset[b + 1] += d->row_offset[b];
  std::vector<RawCluster> sorted((size_t)N);
  {
    std::vector<uint32_t> cur(d->row_offset.begin(), d->row_offset.end() - 1);
    for (const RawCluster& rc : all) sorted[cur[rc.bucket]++] = rc;
  }
  all.clear(); all.shrink_to_fit();
#pragma omp parallel for schedule(dynamic, 16)
  for (int b = 0; b < nb; ++b) {
    std::sort(sorted.begin() + d->row_offset[b], sorted.begin() + d->row_offset[b + 1],
              [](const RawCluster& A, const RawCluster& B) {
                if (A.key != B.key) return A.key < B.key;
                if (A.track != B.track) return A.track < B.track;
                if (A.y != B.y) return A.y < B.y;
                return A.z < B.z;
              });
  }
  d->x.resize(N); d->y.resize(N); d->z.resize(N); d->q.resize(N);
  d->truth_track.resize(N); d->truth_turn.resize(N);
  for (int b = 0; b < nb; ++b) {
    const float xr = (float)c->row_x[b % R];
    for (uint32_t i = d->row_offset[b]; i < d->row_offset[b + 1]; ++i) {
      d->x[i] = xr; d->y[i] = sorted[i].y; d->z[i] = sorted[i].z;
      d->q[i] = (float)(20.0 + 80.0 * ((sorted[i].key >> 20) & 0xFFFF) / 65536.0);   // arbitrary positive charge
      d->truth_track[i] = sorted[i].track; d->truth_turn[i] = sorted[i].turn;
    }
  }
  return d;
}

int64_t tpcgen_n_clusters(const tpcgenData* d) { return d ? (int64_t)d->y.size() : -1; }
int64_t tpcgen_n_tracks(const tpcgenData* d) { return d ? (int64_t)d->t_pt.size() : -1; }

// copy out; any pointer may be NULL
void tpcgen_copy_clusters(const tpcgenData* d, uint32_t* row_offset, float* x, float* y, float* z, float* q,
                          int32_t* truth_track, int32_t* truth_turn) {
  if (row_offset) std::memcpy(row_offset, d->row_offset.data(), d->row_offset.size() * 4);
  size_t nb = d->y.size() * 4;
  if (x) std::memcpy(x, d->x.data(), nb);
  if (y) std::memcpy(y, d->y.data(), nb);
  if (z) std::memcpy(z, d->z.data(), nb);
  if (q) std::memcpy(q, d->q.data(), nb);
  if (truth_track) std::memcpy(truth_track, d->truth_track.data(), nb);
  if (truth_turn) std::memcpy(truth_turn, d->truth_turn.data(), nb);
}
void tpcgen_copy_tracks(const tpcgenData* d, double* pt, double* phi0, double* eta, double* vz, double* zshift,
                        int32_t* charge_sign) {
  size_t nb = d->t_pt.size() * 8;
  if (pt) std::memcpy(pt, d->t_pt.data(), nb);
  if (phi0) std::memcpy(phi0, d->t_phi0.data(), nb);
  if (eta) std::memcpy(eta, d->t_eta.data(), nb);
  if (vz) std::memcpy(vz, d->t_vz.data(), nb);
  if (zshift) std::memcpy(zshift, d->t_zshift.data(), nb);
  if (charge_sign) std::memcpy(charge_sign, d->t_charge_sign.data(), d->t_charge_sign.size() * 4);
}
void tpcgen_free(tpcgenData* d) { delete d; }

}  // extern "C"
