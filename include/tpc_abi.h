/* tpc_abi.h -- C ABI of libtpcgpu.so, the B200 (sm_100a) TPC sector tracker.
 *
 * What the library computes (BASELINE.json north_star; "TPC track finding ... derived
 * from the Run 2 HLT TPC tracking on GPUs"; clusters with single-precision properties in, PAPER.md
 * L69-L70; tracks and the cluster-to-track attachment out):
 *   a1 grid build          per (sector,row) counting sort of the clusters over a (y,z) grid
 *   a2 neighbour finder    best (up,down) pair per cluster against a straight line
 *   a3 cleaner/start hits  reciprocal links only; heads of link chains
 *   a4 tracklet constructor link-chain fit + row-by-row helix Kalman extrapolation (5 params, 15 cov, fp32)
 *   a5 tracklet selector   shared clusters go to the longest / lowest-chi2 tracklet
 *   a6 refit (optional)    Kalman refit of every selected track over its kept clusters: inner and outer state
 *   a7 merger (optional)   links between track segments across row gaps and sector borders
 *   a10 legs (optional)    pairs of track ends that are the two sides of a looper's outer turn
 *   a8 flags (optional)    per cluster: attached / adjacent / protected, removed by rejection strategy A / B
 * The formulas, constants and tie-breaks are DESIGN.md section 3 (readings R0..R27 of SURVEY.md 8(c)).
 *
 * Conventions
 *   - every call returns an int status: TPC_OK (0) or a negative TPC_ERR_*; no exceptions, no global state;
 *   - "DEVICE" pointers are CUDA device pointers of the handle's device, "HOST" pointers are host memory;
 *   - the caller owns every buffer it passes (inputs, outputs, workspace); inputs are never written;
 *   - tpcRun only enqueues work on the given stream and returns; results and the status are valid after
 *     the stream has been synchronised (tpcGetRunStatus does that itself);
 *   - a handle is not thread-safe; distinct handles are independent;
 *   - there is no CPU fallback: without a CUDA device tpcCreate fails with TPC_ERR_CUDA.
 */
#ifndef TPC_ABI_H
#define TPC_ABI_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  TPC_OK = 0,
  TPC_ERR_INVALID_ARG = -1,         /* NULL / negative / inconsistent argument */
  TPC_ERR_UNSORTED_OFFSETS = -2,    /* row_offset not monotone or its ends != 0 / n_clusters (found on the device) */
  TPC_ERR_WORKSPACE_TOO_SMALL = -3,
  TPC_ERR_CAPACITY = -4,            /* an output capacity was exceeded: outputs truncated, nothing written out of
                                       bounds, required sizes are in tpcRunStatus */
  TPC_ERR_CUDA = -5,                /* a CUDA runtime call failed (tpcErrorString gives the last message) */
  TPC_ERR_NONFINITE_INPUT = -6,     /* validate_input was set and a cluster coordinate is NaN/Inf (R25) */
  TPC_ERR_OUT_OF_MEMORY = -7,       /* host allocation of the handle failed */
  TPC_ERR_NOALLOC_LIMIT = -8        /* tpcStartHitsNoAlloc: n_clusters beyond TPC_NOALLOC_MAX_CLUSTERS (nothing was launched) */
};

typedef struct tpcHandle tpcHandle;

/* Detector description (R1, R2).  All pointers HOST, copied by tpcCreate. */
typedef struct {
  int32_t n_sectors;            /* 36 (config 0: 1); 1 <= n_sectors <= 64 */
  int32_t n_rows;               /* 152; 3 <= n_rows <= 255 */
  const float* row_x;           /* [n_rows] local x of the pad-row planes, cm, strictly increasing */
  const float* row_pitch;       /* [n_rows] pad pitch, cm; carried only (may be NULL) */
  const uint8_t* row_dead;      /* [n_rows] 1 = dead row, or NULL */
  float bz_tesla;               /* uniform field, 0.5 */
  float tan_half_sector;        /* tan(10 deg): row half width = row_x * tan_half_sector */
  float z_min, z_max;           /* grid z range, cm; clusters outside are clamped into edge cells */
} tpcGeometry;

/* Table P of DESIGN.md section 3.  tpcDefaultParams fills the defaults given in the comments. */
typedef struct {
  float area_y, area_z;         /* 1.5, 1.5   neighbour window = area * |dx| (O2) */
  float link_dev2_max;          /* 0.64       max squared slope mismatch of a link (O2) */
  float err2_y, err2_z;         /* 0.01, 0.01 measurement variances, cm^2 (O4 Update) */
  float init_var_s, init_var_t, init_var_q;   /* 1, 1, 100  prior variances (O4 step 1) */
  float turn_var_scale;         /* 100        y,z variance scale at the turn (O4 step 4) */
  float max_sinphi;             /* 0.98 */
  float road_sigma, road_min, road_max;       /* 4, 0.3, 2.0  search road (O4 Search) */
  int32_t max_row_gap;          /* 4 */
  int32_t min_chain_hits;       /* 3 */
  int32_t min_tracklet_hits;    /* 10 */
  int32_t min_track_hits;       /* 10 */
  float cell_min, cell_max;     /* 0.5, 8.0   grid cell edge limits, cm (O1; do not change results, R3) */
  float clusters_per_cell;      /* 0.7        target occupancy of a grid cell (implementation choice, R3) */
  int32_t validate_input;       /* 0          1 = scan y,z for NaN/Inf and fail with TPC_ERR_NONFINITE_INPUT */
  int32_t force_wide_keys;      /* 0          1 = use the two-pass selector keys even when the packed 64-bit key
                                              fits (R27; results are identical, for tests) */
  int32_t merge_max_row_gap;    /* 40         O7: rows between the end of a segment and the start of its continuation */
  int32_t merge_back_rows;      /* 5          O7: a continuation in the neighbour sector may start this many rows lower */
  float merge_chi2_max;         /* 50         O7: cut on the diagonal chi2 of a match */
  float tube_radius;            /* 1.5        O8: clusters within this distance of a track are adjacent, cm */
  float inv_pt_protect;         /* 20         O8: tracks with |q/pT| below this (pT > 50 MeV/c) protect */
  int32_t charge_trunc_bits;    /* 4          O9: bits kept after the first non-zero bit of a charge */
  float leg_min_sinphi;         /* 0.5        O10: a refitted track that ends with |sin phi| not below this is a leg end */
  float leg_chi2_max;           /* 50         O10: cut on the diagonal chi2 of the two sides of a turn */
  int32_t leg_max_sectors;      /* 4          O10: the two ends of a turn are at most this many sectors apart (0..8) */
  int32_t leg_max_row_diff;     /* 12         O10: and their last rows at most this many rows */
  float leg_max_centre_dist;    /* 10         O10: and the centres of their circles at most this far apart, cm */
  int32_t pos_bits;             /* 6          O11: positions and residuals are stored in units of 2^-pos_bits cm (0..15) */
  float tube_chi2_max;          /* 0          O8, R49: 0 = the fixed tube alone; > 0: a cluster of the tube must
                                              also have dy^2/(C00+err2_y) + dz^2/(C11+err2_z) <= this (walking state's variances) */
} tpcParams;

/* Input clusters: CSR by (sector,row), fp32 SoA (single-precision cluster properties). */
typedef struct {
  int64_t n_clusters;           /* 0 <= n_clusters < 2^31 */
  const uint32_t* row_offset;   /* DEVICE [n_sectors*n_rows+1]; clusters of (s,r) = [off[s*n_rows+r], off[s*n_rows+r+1]) */
  const float* x;               /* DEVICE [n_clusters] or NULL; not read: a cluster's x is row_x[r] */
  const float* y;               /* DEVICE [n_clusters] local y (pad direction), cm */
  const float* z;               /* DEVICE [n_clusters] z (drift/time direction), cm */
  const float* q;               /* DEVICE [n_clusters] charge or NULL; read only for the optional cl_qcode output */
} tpcClusters;

/* Outputs.  All pointers DEVICE.  Tracks are emitted in ascending tracklet id (= rank of the start hit in
 * ascending global cluster index); a track's clusters in ascending row. */
typedef struct {
  int64_t cap_tracks;           /* capacity of the trk_* arrays */
  int64_t cap_track_clusters;   /* capacity of trk_cl_index */
  int32_t* trk_tracklet;        /* [cap_tracks] tracklet id of the track */
  int32_t* trk_sector;          /* [cap_tracks] */
  int32_t* trk_first_row;       /* [cap_tracks] first / last row with a kept cluster */
  int32_t* trk_last_row;
  int32_t* trk_ncl;             /* [cap_tracks] kept clusters */
  float* trk_x;                 /* [cap_tracks] x of the reference plane (innermost attached row of the tracklet) */
  float* trk_par;               /* [5][cap_tracks] SoA: y, z, sin(phi), dz/ds, q/pT */
  float* trk_cov;               /* [15][cap_tracks] SoA: lower triangle 00,10,11,20,21,22,30,...,44 */
  float* trk_chi2;              /* [cap_tracks] chi2 of the constructor's down pass (R22: not refitted) */
  uint32_t* trk_cl_offset;      /* [cap_tracks+1] CSR offsets into trk_cl_index */
  uint32_t* trk_cl_index;       /* [cap_track_clusters] global (input) cluster indices */
  /* optional per-stage outputs for parity tests; any may be NULL */
  int32_t* link_up_raw;         /* [n_clusters] O2 links as global input indices, -1 = none */
  int32_t* link_dn_raw;
  int32_t* link_up;             /* [n_clusters] O3 cleaned links */
  int32_t* link_dn;
  uint32_t* start_hits;         /* [cap_tracklets] O3 start hits, ascending global index */
  int32_t* tl_status;           /* [cap_tracklets] 0 discarded in the chain fit, 1 rejected, 2 accepted */
  int32_t* tl_nhits;            /* [cap_tracklets] */
  int32_t* tl_first_row;        /* [cap_tracklets] */
  int32_t* tl_last_row;
  int32_t* tl_rowhit;           /* [cap_tracklets][n_rows] global input indices / -1 (tracklet-major) */
  float* tl_x;                  /* [cap_tracklets] */
  float* tl_par;                /* [cap_tracklets][5] (tracklet-major) */
  float* tl_cov;                /* [cap_tracklets][15] */
  float* tl_chi2;               /* [cap_tracklets] */
  /* optional O6 refit of the selected tracks over their kept clusters (DESIGN.md section 3 "O6"; the paper names a
   * track refit at PAPER.md L11 / L92).  All NULL = no refit; otherwise ALL eight must be given.  Never changes trk_*. */
  int32_t* trk_rf_status;       /* [cap_tracks] 1 = refitted, 0 = a Propagate / Update was refused (outputs zero) */
  float* trk_rf_x_in;           /* [cap_tracks] x of the first kept cluster: reference plane of the inner state */
  float* trk_rf_par_in;         /* [5][cap_tracks] inner state (after the down pass) */
  float* trk_rf_cov_in;         /* [15][cap_tracks] */
  float* trk_rf_chi2;           /* [cap_tracks] chi2 of the down pass, ndf = 2 ncl - 5 */
  float* trk_rf_x_out;          /* [cap_tracks] x of the last kept cluster: reference plane of the outer state */
  float* trk_rf_par_out;        /* [5][cap_tracks] outer state (after the up pass) */
  float* trk_rf_cov_out;        /* [15][cap_tracks] */
  /* optional O7 links between track segments (DESIGN.md section 3 "O7").  All NULL = no merger; otherwise
   * ALL four must be given together with the refit outputs (the merger works on the refitted states). */
  int32_t* trk_mg_next;         /* [cap_tracks] track that continues this one, -1 none */
  int32_t* trk_mg_prev;         /* [cap_tracks] track this one continues, -1 none */
  int32_t* trk_mg_head;         /* [cap_tracks] first track of the chain (itself if unlinked) */
  float* trk_mg_chi2;           /* [cap_tracks] chi2 of the link to trk_mg_next, 0 if none */
  /* optional O10 pairs of looper legs (DESIGN.md section 3 "O10").  Both NULL = none; otherwise both,
   * together with the refit outputs (the outer states are compared). */
  int32_t* trk_leg_partner;     /* [cap_tracks] the track whose outer end is the other side of this track's outer turn, -1 none;
                                   partner[partner[k]] == k */
  float* trk_leg_chi2;          /* [cap_tracks] chi2 of that pair (the same on both), 0 if none */
  /* optional O8 per-cluster flags (DESIGN.md section 3 "O8").  Both NULL = none; otherwise both, together
   * with the refit outputs.  Indexed by the INPUT cluster index. */
  uint8_t* cl_flags;            /* [n_clusters] 1 attached, 2 adjacent, 4 protected, 8 removed by strategy A, 16 by strategy B */
  int32_t* cl_owner;            /* [n_clusters] track with the cluster in its tube (highest momentum), -1 none */
  float* cl_res_y;              /* [n_clusters] optional with the two above (both or none): track-model residuals */
  float* cl_res_z;              /*   y_c - y_track, z_c - z_track of the clusters attached to refitted tracks, 0 elsewhere */
  /* optional O9 dynamic-precision charge code (DESIGN.md section 3 "O9"); needs tpcClusters.q */
  uint16_t* cl_qcode;           /* [n_clusters] integer charge with all bits beyond charge_trunc_bits after the first
                                   non-zero bit rounded away; NULL = not computed */
  /* optional O11 16-bit integer format (DESIGN.md section 3 "O11"): y16 | z16 << 16 per cluster, v16 = the
   * integer nearest to v * 2^pos_bits (ties to even), saturated to [-32768, 32767] */
  uint32_t* cl_pos_code;        /* [n_clusters] code of the absolute (y, z) of every cluster; NULL = not computed */
  uint32_t* cl_res_code;        /* [n_clusters] code of the track-model residuals (0 where there is none); needs cl_flags and
                                   cl_owner (and with them the refit outputs); NULL = not computed */
  /* optional O12 merged tracks and leg labels (DESIGN.md section 3 "O12", R46..R48); all four or
   * none; need the merger and the leg-pair outputs.  When they are given together with cl_flags, the cluster flags treat
   * secondary legs as not protecting and their clusters as removable by strategy A (L86). */
  int32_t* trk_mt_id;           /* [cap_tracks] the merged track of every track: the smallest head index of its one or two legs */
  int32_t* trk_mt_rank;         /* [cap_tracks] 0 = on the primary (first) leg of its merged track, 1 = on the secondary leg */
  uint32_t* mt_cl_offset;       /* [cap_tracks + 1] cluster list of the merged track named by track k: [off[k], off[k+1]);
                                   empty for tracks that name none */
  uint32_t* mt_cl_index;        /* [cap_track_clusters] clusters in the order along the particle's path: the primary leg from
                                   its inner end outwards, then the secondary leg from the turn inwards */
} tpcTracks;

/* Filled by tpcGetRunStatus after the stream has drained. */
typedef struct {
  int32_t status;               /* TPC_OK, TPC_ERR_CAPACITY, TPC_ERR_UNSORTED_OFFSETS, TPC_ERR_NONFINITE_INPUT */
  int32_t kernel_launches;      /* kernels + memsets enqueued by the last tpcRun */
  int64_t n_clusters;
  int64_t n_start_hits;         /* = tracklet ids; required cap_tracklets */
  int64_t n_tracklets;          /* accepted tracklets (status 2) */
  int64_t n_tracklet_hits;      /* H: hits summed over accepted tracklets */
  int64_t n_tracks;             /* required cap_tracks */
  int64_t n_track_clusters;     /* required cap_track_clusters */
  int64_t n_cells;              /* grid cells over all (sector,row) */
  float stage_ms[8];            /* per-stage device times of the last tpcRun / tpcRunHost when profiling is on (else 0;
                                   always 0 from tpcCollectHost: the stage events belong to the handle, not to a slot):
                                   0 grid, 1 neighbour finder, 2 cleaner+start hits, 3 constructor, 4 selector,
                                   5 optional refit, merger and exports, 6 total, 7 refit alone */
  float merge_ms;               /* the O7 merger alone (profiling on, merger requested) */
  float pack_ms;                /* the O9 charge code and the O11 position code alone (profiling on, cl_qcode / cl_pos_code requested) */
  float flags_ms;               /* the O8 cluster flags alone (profiling on, flags requested) */
  float legs_ms;                /* the O10 leg pairs alone (profiling on, legs requested) */
  float merged_ms;              /* the O12 merged tracks alone (profiling on, merged tracks requested) */
  float submit_ms[2];           /* tpcCollectHost only: device time of the slot from its first copy in to the end of its
                                   kernels [0] and to the end of its copies out [1] (includes waiting for the other slot) */
} tpcRunStatus;

int tpcDefaultParams(tpcParams* p);

/* Creates a tracker on CUDA device `cuda_device`; copies geometry and parameters.  HOST pointers. */
int tpcCreate(tpcHandle** out, const tpcGeometry* g, const tpcParams* p, int cuda_device);
int tpcDestroy(tpcHandle* h);

/* Bytes of DEVICE workspace tpcRun needs for up to n_clusters clusters and cap_tracklets start hits. */
int tpcWorkspaceBytes(const tpcHandle* h, int64_t n_clusters, int64_t cap_tracklets, size_t* bytes);

/* Enqueues a1..a5 on `cuda_stream` (a cudaStream_t, NULL = default stream) and returns without synchronising.
 * `workspace` is DEVICE memory of at least tpcWorkspaceBytes(n_clusters, cap_tracklets), 256-byte aligned.
 * Argument errors are returned here; data-dependent errors (capacity, offsets) by tpcGetRunStatus. */
int tpcRun(tpcHandle* h, const tpcClusters* in, tpcTracks* out, int64_t cap_tracklets, void* workspace,
           size_t workspace_bytes, void* cuda_stream);

/* Synchronises with the last tpcRun and reports counts, required capacities and the data-dependent status. */
int tpcGetRunStatus(tpcHandle* h, tpcRunStatus* out);

/* 1 = record CUDA events between the stages of every tpcRun (stage_ms); 0 = off (default). */
int tpcSetProfiling(tpcHandle* h, int on);

/* Host-buffer convenience call (the end-to-end path a host application uses): copies row_offset, y, z
 * (HOST, pageable or pinned) to device memory owned by the handle (grown on demand), runs a1..a5, copies
 * the tracks back into the HOST arrays of `out_host` (same layout as tpcTracks but HOST pointers; the
 * optional per-stage pointers must be NULL) and synchronises.  *status receives the run status. */
int tpcRunHost(tpcHandle* h, int64_t n_clusters, const uint32_t* row_offset, const float* y, const float* z,
               tpcTracks* out_host, tpcRunStatus* status, void* cuda_stream);

/* Double-buffered form of tpcRunHost for a stream of events: tpcSubmitHost(slot) enqueues the copies in, a1..a5 and
 * the copies out of one event on the slot's own stream and returns at once; tpcCollectHost(slot) waits for it and
 * reports its status.  slot is 0 or 1, so that the copies of one event overlap the kernels of the other.  The HOST
 * buffers (inputs and the arrays of `out_host`, pinned for real overlap) must stay valid and untouched until the
 * collect.  The counts are not known at submit time: up to min(capacity of the handle's device buffers, capacity of
 * out_host) entries are copied back and tpcRunStatus says how many are valid.  status TPC_ERR_CAPACITY = a capacity
 * was too small (first events of a stream): run that event again with tpcRunHost, which grows the buffers.  The device
 * pools of a slot grow with cudaFree / cudaMalloc, which synchronise the device: a submit that has to grow its pools (the
 * first events of a stream, or an event larger than any before) waits for the other slot's event; steady state allocates
 * nothing. */
int tpcSubmitHost(tpcHandle* h, int slot, int64_t n_clusters, const uint32_t* row_offset, const float* y, const float* z,
                  const tpcTracks* out_host);
int tpcCollectHost(tpcHandle* h, int slot, tpcRunStatus* status);

const char* tpcErrorString(int code);
const char* tpcLastCudaError(const tpcHandle* h);

/* Diagnostic: the Kalman update divides six numerators by one denominator with a shared reciprocal (csrc/tpc_kalman.cuh,
 * `divShared`), which must be bit-identical to the IEEE division the formula sheet writes (R0).  This call runs
 * both forms on the device for n_threads x 48 operand pairs drawn over the whole domain of the shared form (seeded,
 * edge values included) and reports how many were tested and how many bit patterns differ (must be 0).  Synchronous. */
int tpcSelfTestDivision(tpcHandle* h, int64_t n_threads, uint64_t seed, int64_t* n_tested, int64_t* n_mismatches);

/* ---- the allocation-free entry point (csrc/tpc_noalloc.cu) ---------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the a3 start-hit list (O3, R8) computed with NO workspace argument and no
 * allocation of any kind.  The scratch of its stream compaction (one count per 2048 clusters) is a static device array
 * of the library: 33 024 bytes that every GPU which loads libtpcgpu.so holds until the process exits.  That fixes the
 * largest input: */
#define TPC_NOALLOC_MAX_CLUSTERS 16777216 /* 2^24; more -> TPC_ERR_NOALLOC_LIMIT */

/* The limit again, for callers that cannot read the macro (ctypes). */
int64_t tpcNoAllocMaxClusters(void);

/* Looks up the device address of the static scratch on `cuda_device` (once per device; idempotent, thread-safe).
 * tpcStartHitsNoAlloc does this itself on its first call for a device; call it beforehand where the first call would be
 * inside a stream capture (the look-up is not a stream operation and may be refused there). */
int tpcNoAllocSetup(int cuda_device);

/* Enqueues three kernels on `cuda_stream` (a cudaStream_t, NULL = default stream) of `cuda_device` and returns without
 * synchronising; calls no cudaMalloc / cudaFree / allocating routine.
 *   link_up, link_dn  DEVICE [n_clusters] cleaned links as global input indices, -1 = none (the tpcTracks.link_up /
 *                     link_dn outputs of tpcRun); read only; 0 <= n_clusters <= TPC_NOALLOC_MAX_CLUSTERS
 *   start_hits        DEVICE [cap_start_hits] out: global input indices c with link_dn[c] == -1 and link_up[c] != -1,
 *                     ascending (= tpcTracks.start_hits); entries beyond cap_start_hits are not written
 *   n_start_hits      DEVICE [1] out: the number of start hits found (the required cap_start_hits, also when truncated)
 * Outputs are valid once the stream has drained.  Argument errors (TPC_ERR_INVALID_ARG, TPC_ERR_NOALLOC_LIMIT) and
 * launch errors (TPC_ERR_CUDA) are returned here; tpcNoAllocLastError gives the text.
 * ALL calls on a device share the one scratch array: calls that overlap on the GPU (different streams without an
 * ordering between them, graphs in flight together) race and give wrong lists; calls ordered on the device (one
 * stream, or events between streams) are safe.  The array keeps the last call's contents; no call relies on them. */
int tpcStartHitsNoAlloc(int cuda_device, int64_t n_clusters, const int32_t* link_up, const int32_t* link_dn,
                        uint32_t* start_hits, int64_t cap_start_hits, int64_t* n_start_hits, void* cuda_stream);

/* Text of the last error of the two calls above on this host thread ("" after a success). */
const char* tpcNoAllocLastError(void);

#ifdef __cplusplus
}
#endif
#endif /* TPC_ABI_H */
