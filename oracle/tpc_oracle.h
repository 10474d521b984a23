/* tpc_oracle.h -- C interface of the CPU ORACLE of the TPC sector tracker.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this library.  It shares no code, header, table or
 * constant with the CUDA path (paper_1910_12214_b200/csrc, include/tpc_abi.h); the structs below are
 * the oracle's own.
 *
 * What it computes: the five steps O1..O5 of DESIGN.md section 3 (formula sheet), which restates
 * the reading of BASELINE.json north_star adopted because PAPER.md gives
 * no algorithmic detail for the tracker ("derived from the Run 2 HLT GPU
 * tracker", nothing more).  Single thread, plain loops, one rounding per written operation, no FMA
 * contraction (build with -ffp-contract=off -fno-fast-math), binary32 (the parity reference) or
 * binary64 (algebra checks).
 *
 * Pins (tests/test_oracle_*.py): grid search == brute-force search; collinear / hand-built link
 * cases; reciprocity and path invariants; Propagate vs the closed-form asin helix and vs finite
 * differences; Update / fit vs numpy least squares; exact helix recovery; unit pulls; full
 * attachment of noise-free high-pT helices; Search (road widths, clamps, nearest, ties) and the gap / length rules of
 * O4 / O5 on hand-worked cases; selector vs sorted greedy; O6..O10: see DESIGN.md, pins table.
 * Parity unpinned: physics efficiency / fake rate on configs 1-4 (no reference numbers exist).
 */
#ifndef TPC_ORACLE_H
#define TPC_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int32_t n_sectors, n_rows;
  const float* row_x;        /* [n_rows] */
  const uint8_t* row_dead;   /* [n_rows] or NULL */
  float bz_tesla, tan_half_sector, z_min, z_max;
} orcGeometry;

/* Table P of SURVEY.md 8(c) / DESIGN.md 3; orcDefaultParams fills the defaults */
typedef struct {
  float area_y, area_z, link_dev2_max;
  float err2_y, err2_z, init_var_s, init_var_t, init_var_q, turn_var_scale;
  float max_sinphi, road_sigma, road_min, road_max;
  int32_t max_row_gap, min_chain_hits, min_tracklet_hits, min_track_hits;
  float cell_min, cell_max;
  int32_t merge_max_row_gap, merge_back_rows;   /* O7: 40, 5 */
  float merge_chi2_max;                         /* O7: 50 */
  float tube_radius, inv_pt_protect;            /* O8: 1.5 cm, 20 c/GeV (pT = 50 MeV/c) */
  float leg_min_sinphi, leg_chi2_max;           /* O10: 0.5, 50 */
  int32_t leg_max_sectors, leg_max_row_diff;    /* O10: 4, 12 */
  float leg_max_centre_dist;                    /* O10: 10 cm */
  float tube_chi2_max;                          /* O8, R49: 0 = fixed tube only; > 0: also dy^2/(C00+err2_y) + dz^2/(C11+err2_z) <= this */
} orcParams;

typedef struct orcResult orcResult;

enum { ORC_OK = 0, ORC_ERR_INVALID_ARG = -1, ORC_ERR_UNSORTED_OFFSETS = -2 };
enum { ORC_BRUTE_FORCE = 1, ORC_FP64 = 2, ORC_REFIT = 4, ORC_MERGE = 8 /* implies ORC_REFIT */,
       ORC_FLAGS = 16 /* implies ORC_REFIT */, ORC_LEGS = 32 /* implies ORC_REFIT */,
       ORC_MERGED = 64 /* implies ORC_MERGE and ORC_LEGS */ };

void orcDefaultParams(orcParams* p);

/* Runs O1..O5 on host arrays.  flags: ORC_BRUTE_FORCE = every search loops over all clusters of the
 * row instead of the grid; ORC_FP64 = all arithmetic in binary64.  On success *out owns the result. */
int orcRun(const orcGeometry* g, const orcParams* p, int64_t n_clusters, const uint32_t* row_offset,
           const float* y, const float* z, int flags, orcResult** out);
void orcFree(orcResult* r);

/* sizes */
int64_t orcNumClusters(const orcResult*);
int64_t orcNumStartHits(const orcResult*);   /* == number of tracklet ids */
int64_t orcNumTracks(const orcResult*);
int64_t orcNumTrackClusters(const orcResult*);

/* O1: grid invariants. sorted_to_orig [n]; cell_of_sorted [n] (cell id inside the bucket);
 * n_cells [n_sectors*n_rows]. NULL-able. Empty when ORC_BRUTE_FORCE. */
void orcGetGrid(const orcResult*, uint32_t* sorted_to_orig, int32_t* cell_of_sorted, int32_t* n_cells);
/* O2/O3: links, global original indices, -1 none */
void orcGetLinks(const orcResult*, int32_t* up_raw, int32_t* dn_raw, int32_t* up, int32_t* dn);
void orcGetStartHits(const orcResult*, uint32_t* start_hits);
/* How often O4 ran Propagate, Update, Search, and how many clusters its Searches found inside their roads (four counts):
 * the algorithmic operation count of the measurement. */
void orcGetO4Counts(const orcResult*, int64_t* four);
/* The same for O2: clusters that have both a row above and a row below, their up candidates, their down candidates and
 * the (u, d) pairs the definition evaluates (sum of nU * nD). */
void orcGetO2Counts(const orcResult*, int64_t* four);
/* O4: one entry per start hit (tracklet id = rank).  status: 0 discarded in the chain fit,
 * 1 built but rejected (nhits < min_tracklet_hits or no snapshot), 2 accepted.
 * rowhit [n_start*n_rows] global indices / -1; x [n_start]; par [n_start*5]; cov [n_start*15]. */
void orcGetTracklets(const orcResult*, int32_t* status, int32_t* nhits, int32_t* first_row, int32_t* last_row,
                     int32_t* rowhit, double* x, double* par, double* cov, double* chi2);
/* O5: tracks in ascending tracklet id; par [n_tracks*5], cov [n_tracks*15] (track-major);
 * cl_offset [n_tracks+1]; cl_index [n_track_clusters] ascending row. */
void orcGetTracks(const orcResult*, int32_t* tracklet_id, int32_t* sector, int32_t* first_row, int32_t* last_row,
                  int32_t* ncl, double* x, double* par, double* cov, double* chi2, uint32_t* cl_offset,
                  uint32_t* cl_index);

/* O6 (NEXT-2 of SURVEY.md 8(f), DESIGN.md section 3 "O6"): refit of every selected track over its kept clusters,
 * only when orcRun was called with ORC_REFIT.  status [n_tracks] 1 = refitted, 0 = Propagate / Update refused;
 * *_in = state at the first kept cluster after the down pass (chi2 of that pass), *_out = state at the last kept
 * cluster after the up pass.  par [n_tracks*5], cov [n_tracks*15] track-major.  Pins: tests/test_oracle_refit.py. */
void orcGetRefit(const orcResult*, int32_t* status, double* x_in, double* par_in, double* cov_in, double* chi2,
                 double* x_out, double* par_out, double* cov_out);
/* The same refit on n given clusters of one sector (rows ascending, binary64 coordinates kept exact when fp64):
 * inner22 / outer22 = x, y, z, s, t, q, C[15], chi2.  Returns 1 on success. */
int orcRefitPoints(const orcGeometry* g, const orcParams* p, int n, const int32_t* rows, const double* y, const double* z,
                   int fp64, double* inner22, double* outer22);

/* O7 (NEXT-1 of SURVEY.md 8(f), DESIGN.md section 3 "O7"): links between track segments, only with ORC_MERGE.
 * next / prev / head [n_tracks] track indices (-1 none; head = first track of the chain), chi2 [n_tracks] of the link
 * to next (0 if none).  Pins: tests/test_oracle_merge.py. */
void orcGetMerge(const orcResult*, int32_t* next, int32_t* prev, int32_t* head, double* chi2);
/* O8 (NEXT-3 of SURVEY.md 8(f), DESIGN.md section 3 "O8"): per-cluster flags, only with ORC_FLAGS.
 * flags [n_clusters] bit mask 1 attached, 2 adjacent, 4 protected (some track with pT > 50 MeV/c, |phi| < 70 degrees on that
 * row and not a secondary leg has the cluster in its tube), 8 removed by strategy A, 16 removed by strategy B;
 * owner [n_clusters] track index of the highest-momentum track with the cluster in its tube, -1 none. */
void orcGetClusterFlags(const orcResult*, uint8_t* flags, int32_t* owner);
/* track-model residuals (O8, R39) of the clusters attached to refitted tracks, 0 elsewhere;
 * only with ORC_FLAGS.  res_y, res_z [n_clusters]. */
void orcGetResiduals(const orcResult*, double* res_y, double* res_z);

/* O9 (part of NEXT-4, DESIGN.md section 3 "O9"): dynamic-precision code of n_values charges: the integer
 * nearest to q, with every bit more than trunc_bits after its first non-zero bit rounded away.  Returns 0 on bad arguments. */
int orcPackCharge(int64_t n_values, const float* q, int trunc_bits, uint16_t* code);

/* O11 (rest of NEXT-4, DESIGN.md section 3 "O11"): 16-bit integer format of positions (absolute, or
 * residuals to the track model): code[i] = y16 | z16 << 16 with v16 = the integer nearest to v * 2^bits (ties to even),
 * saturated to [-32768, 32767], NaN -> 0.  Returns 0 on bad arguments. */
int orcPackPositions(int64_t n_values, const float* y, const float* z, int bits, uint32_t* code);

/* Pieces of O7 for the pins.  state = {x, y, z, s, t, q}, cov = 15 lower-triangle elements, in/out as doubles.
 * orcRotate: frame turned by alpha (radians); returns 1 on success, 0 (untouched) on failure.
 * orcMatch: chi2 of the match of outer state a to inner state b (b at plane b_state[0]); rel = 0 same sector,
 * +1 / -1 b in the next / previous sector; returns 1 and *chi2 when admissible (chi2 <= merge_chi2_max), else 0. */
int orcRotate(double* state, double* cov, double alpha, double bz_tesla, double max_sinphi, int fp64);
int orcMatch(const orcParams* p, double bz_tesla, const double* a_state, const double* a_cov, int rel,
             const double* b_state, const double* b_cov, int fp64, double* chi2);

/* O10 (rest of NEXT-1, DESIGN.md section 3 "O10"; legs of loopers): the two sides of a turn,
 * only with ORC_LEGS.  partner [n_tracks] = the track whose outer end is the other side of this track's outer turn
 * (-1 none; partner[partner[k]] == k), chi2 [n_tracks] of that pair (0 if none).  Pins: tests/test_oracle_legs.py. */
void orcGetLegs(const orcResult*, int32_t* partner, double* chi2);
/* O12 (rest of NEXT-1 and what NEXT-3 needs of it; DESIGN.md section 3 "O12", readings R46..R48; "only the
 * primary, first leg is protected", L86, L92 "merging of track segments and legs of the same track"): merged tracks, only
 * with ORC_MERGED.  id [n_tracks] = the merged track of every track (the smallest head index of its one or two legs),
 * rank [n_tracks] 0 = on the primary (first) leg, 1 = on the secondary leg; cl_offset [n_tracks + 1], cl_index
 * [n_track_clusters]: cluster list of the merged track in the order along the particle's path, stored at the index of the
 * track that names it (empty ranges elsewhere).  With ORC_FLAGS | ORC_MERGED the cluster flags treat secondary legs as
 * not protecting and their clusters as removable by strategy A (L86).  Pins: tests/test_oracle_merged.py. */
void orcGetMerged(const orcResult*, int32_t* id, int32_t* rank, uint32_t* cl_offset, uint32_t* cl_index);
/* Pieces of O10 for the pins.  orcMirror: the state seen from the frame turned by 180 degrees and walked backwards.
 * orcLegMatch: chi2 of two outer states a, b (b's sector d sectors after a's); returns 1 and *chi2 when admissible. */
void orcMirror(double* state, double* cov);
int orcLegMatch(const orcParams* p, double bz_tesla, const double* a_state, const double* a_cov, int d,
                const double* b_state, const double* b_cov, int fp64, double* chi2);

/* Single KF steps for the pins.  state = {x, y, z, s, t, q}, cov = 15 lower-triangle elements
 * (00,10,11,20,21,22,30,...,44), both in/out as doubles (rounded to binary32 first unless fp64).
 * Return 1 on success, 0 on failure (state untouched). */
int orcPropagate(double* state, double* cov, double x_new, double bz_tesla, double max_sinphi, int fp64);
/* One Search of O4 (DESIGN.md section 3 "Search", reading R13) for the pins: the n given clusters of one sector
 * (rows ascending, index = position in the arrays) are the whole input; the road is taken from the state
 * {x, y, z, s, t, q} and its covariance, on pad row `row`.  Returns the index of the picked cluster, -1 when the
 * road is empty, -2 on bad arguments.  brute = 1: every cluster of the row is tested, no grid. */
int orcSearch(const orcGeometry* g, const orcParams* p, int n, const int32_t* rows, const float* y, const float* z, int row,
              const double* state, const double* cov, int fp64, int brute);

int orcUpdate(double* state, double* cov, double* chi2, double ym, double zm, double err2_y, double err2_z, int fp64);

#ifdef __cplusplus
}
#endif
#endif
