// tpc_api.cu -- host side of libtpcgpu.so: the C ABI of include/tpc_abi.h, workspace layout and the launch
// sequence a1..a5 on one stream (no host round trip inside tpcRun).
//
// Build (see paper_1910_12214_b200/build.py):
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo --fmad=false -prec-div=true -prec-sqrt=true
//        -ftz=false -shared -Xcompiler -fPIC tpc_api.cu -o libtpcgpu.so
#include "../../include/tpc_abi.h"

#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "tpc_common.cuh"
#include "tpc_scan.cuh"
#include "tpc_grid.cuh"
#include "tpc_links.cuh"
#include "tpc_kalman.cuh"
#include "tpc_tracklet.cuh"
#include "tpc_select.cuh"
#include "tpc_refit.cuh"
#include "tpc_merge.cuh"
#include "tpc_legs.cuh"
#include "tpc_flags.cuh"
#include "tpc_merged.cuh"

using namespace tpc;

namespace {

constexpr size_t ALIGN = 256;
inline size_t alignUp(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }
inline int64_t ceilDiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

struct Workspace {
  GridDesc* desc;
  uint32_t* chunk_base;      // [nb+1] first neighbour-finder CTA of every bucket
  uint32_t* chunk_bucket;    // [ceil(N/128)+nb] bucket of every neighbour-finder CTA
  uint4* chunk_reg;          // [ceil(N/128)+nb][2] per neighbour-finder CTA: candidate ranges (kD0, kD1, kU0, kU1); (first cluster, bucket end, bucket, -)
  uint32_t* cell_start;
  uint32_t* rank;            // aliases spos_by_orig (a1 only)
  float2* syz;
  uint32_t* s2o;
  int32_t *lup, *ldn, *cup, *cdn;
  int32_t* spos_by_orig;
  uint32_t* tiles32;         // tile sums: cells scan / start compaction
  unsigned long long* tiles64;
  uint32_t *start_orig, *start_pos;
  SeedRec* work_list;        // long seeds, in the order the constructor takes them
  TurnRec* turn_list;        // [capT] constructUp -> constructDown<0>
  uint4* down_list;          // [capT][DOWNREC_WORDS / 4] constructDown<0> -> constructDown<1>
  uint32_t* gap_idx;         // [capT] work-list indices of the seeds with a gap row in their span
  TrackletStore tl;
  unsigned long long *tsel, *tscan;
  int32_t *kept_first, *kept_last;
  unsigned long long* owner_key;
  uint32_t* owner_id;
  uint32_t *mg_start, *mg_fill, *mg_list;   // merger: tracks bucketed by (sector, first row, dip bin)
  uint32_t *mg_ostart, *mg_ofill, *mg_order;   // the same buckets over the outer states: the order mergeMatch works in
  float4* mg_rec;            // [capT] dip, curvature and their variances of the inner states, in list order
  uint32_t* mg_maxv;         // [n_buckets] largest binned dip variance of a (sector, row)
  uint32_t* mg_tiles;        // tile sums of the bucket scan
  uint32_t *rf_hist, *rf_fill, *rf_order;   // refit: tracks ordered by length
  int32_t* mg_best_b;
  float* mg_chi_b;
  unsigned long long* mg_key_a;
  unsigned long long* fl_key;      // [N] bids of the cluster flags
  uint32_t* fl_prot;               // [ceil(N / 32)] protection bits of the cluster flags
  uint32_t* mt_tiles;              // tile sums of the merged-track offsets scan
  uint32_t *lg_start, *lg_fill, *lg_list;   // leg pairs: leg ends bucketed by (sector, sign, last row, dip bin)
  float4* lg_rec;                           // [capT] dip, curvature and their variances of the leg ends, in list order
  uint32_t *lg_maxv, *lg_tiles;             // largest dip variance per (sector, sign, row); tile sums of the bucket scan
  int32_t* lg_best;
  float* lg_chi;
  size_t bytes;
};

}  // namespace

struct tpcHandle {
  int device = 0;
  tpcParams params{};
  DevParams P{};
  std::vector<float> row_x;
  float* d_row_x = nullptr;
  int16_t *d_up = nullptr, *d_dn = nullptr;
  uint8_t* d_dead = nullptr;
  int64_t* d_cnt = nullptr;        // CNT_COUNT counters + 1 slot for the packed selector total
  int64_t* h_cnt = nullptr;        // pinned copy
  cudaEvent_t ev_done = nullptr;
  cudaEvent_t ev_stage[19] = {};   // ... 13/14 around the charge code, 15/16 leg pairs, 17/18 merged tracks
  //   // 0..6 stage boundaries, 7/8 around the optional refit, 9/10 merger, 11/12 flags
  int profiling = 0;
  int launches = 0;
  int gb_smem_cells = 24 * 1024;      // cells of a bucket whose histogram gridBuild keeps in shared memory (96 KB)
  int gb_smem_bytes = 220 * 1024;     // dynamic shared memory of gridBuild: the histogram and, behind it, the stage of the scatter
  int tc_grid[4] = {148, 148, 148, 148};   // persistent grids of the constructor passes: SMs x resident blocks
  bool pending = false;
  int64_t last_n = 0;
  double cells_per_bucket_bound = 0;   // sum over buckets of the n-independent part of the cell bound
  char cuda_msg[256] = {0};
  // pools of tpcRunHost
  void* pool[16] = {};
  size_t pool_bytes[16] = {};
  int64_t hint_T = 0, hint_K = 0, hint_C = 0;   // capacities the last tpcRunHost needed (+ head-room)
  // The per-run state above (d_cnt, h_cnt, ev_done, launches, pending, last_n, pool, pool_bytes) is the ACTIVE slot's;
  // tpcSubmitHost / tpcCollectHost keep two more copies of it (double buffering) and swap them in and out.
  struct Slot {
    bool init = false;
    int64_t* d_cnt = nullptr; int64_t* h_cnt = nullptr; cudaEvent_t ev_done = nullptr;
    int launches = 0; bool pending = false; int64_t last_n = 0;
    void* pool[16] = {}; size_t pool_bytes[16] = {};
    cudaStream_t stream = nullptr;
    cudaEvent_t ev_begin = nullptr, ev_kernels = nullptr;   // first copy in / end of the kernels of the submitted run
    bool submitted = false;
    int64_t capK = 0, capC = 0;      // device capacities of the submitted run
    tpcTracks oh{};                  // host outputs of the submitted run
  } slots[3];
  int cur_slot = 0;
};

namespace {

int cudaFail(tpcHandle* h, cudaError_t e, const char* what) {
  if (h) snprintf(h->cuda_msg, sizeof(h->cuda_msg), "%s: %s", what, cudaGetErrorString(e));
  return TPC_ERR_CUDA;
}
// after every kernel launch of tpcRun: count it, and name the kernel if the launch itself was refused
#define TPC_LAUNCHED(name)                                                     \
  do {                                                                         \
    ++L;                                                                       \
    const cudaError_t e_ = cudaPeekAtLastError();                              \
    if (e_ != cudaSuccess) { cudaGetLastError(); return cudaFail(h, e_, "launch of " name); } \
  } while (0)
#define TPC_CUDA(h, call)                                   \
  do {                                                      \
    cudaError_t e_ = (call);                                \
    if (e_ != cudaSuccess) return cudaFail(h, e_, #call);   \
  } while (0)

int64_t capCells(const tpcHandle* h, int64_t n) {
  const double cpc = h->params.clusters_per_cell;
  return (int64_t)((double)n / cpc * 1.01 + h->cells_per_bucket_bound * 1.01) + 4 * h->P.n_buckets + 1024;
}

// carve the workspace; base may be NULL (size query)
Workspace layout(const tpcHandle* h, int64_t N, int64_t capT, char* base) {
  Workspace w{};
  size_t o = 0;
  auto take = [&](size_t bytes) { char* p = base ? base + o : nullptr; o += alignUp(bytes); return (void*)p; };
  const int nb = h->P.n_buckets, R = h->P.n_rows;
  const int64_t cc = capCells(h, N);
  const int64_t Nn = N > 0 ? N : 1, Tn = capT > 0 ? capT : 1;
  w.desc = (GridDesc*)take(sizeof(GridDesc) * nb);
  w.chunk_base = (uint32_t*)take(4 * (size_t)(nb + 1));
  w.chunk_bucket = (uint32_t*)take(4 * (size_t)(ceilDiv(Nn, NF_THREADS) + nb));
  w.chunk_reg = (uint4*)take(32 * (size_t)(ceilDiv(Nn, NF_THREADS) + nb));
  w.cell_start = (uint32_t*)take(4 * (size_t)(cc + 1));
  w.spos_by_orig = (int32_t*)take(4 * (size_t)Nn);
  w.rank = (uint32_t*)w.spos_by_orig;
  w.syz = (float2*)take(8 * (size_t)Nn);
  w.s2o = (uint32_t*)take(4 * (size_t)Nn);
  w.lup = (int32_t*)take(4 * (size_t)Nn);
  w.ldn = (int32_t*)take(4 * (size_t)Nn);
  w.cup = (int32_t*)take(4 * (size_t)Nn);
  w.cdn = (int32_t*)take(4 * (size_t)Nn);
  const int64_t t32 = ceilDiv(cc + 1, SCAN_TILE) + ceilDiv(Nn, CP_TILE) + 2;
  w.tiles32 = (uint32_t*)take(4 * (size_t)t32);
  w.tiles64 = (unsigned long long*)take(8 * (size_t)(ceilDiv(Tn, SCAN_TILE) + 2));
  w.start_orig = (uint32_t*)take(4 * (size_t)Tn);
  w.start_pos = (uint32_t*)take(4 * (size_t)Tn);
  w.work_list = (SeedRec*)take(sizeof(SeedRec) * (size_t)Tn);
  w.turn_list = (TurnRec*)take(sizeof(TurnRec) * (size_t)Tn);
  w.down_list = (uint4*)take(4 * (size_t)DOWNREC_WORDS * (size_t)Tn);
  w.gap_idx = (uint32_t*)take(4 * (size_t)Tn);
  w.tl.capT = capT;
  w.tl.n_rows = R;
  w.tl.status = (int32_t*)take(4 * (size_t)Tn);
  w.tl.nhits = (int32_t*)take(4 * (size_t)Tn);
  w.tl.first_row = (int32_t*)take(4 * (size_t)Tn);
  w.tl.last_row = (int32_t*)take(4 * (size_t)Tn);
  w.tl.sector = (int32_t*)take(4 * (size_t)Tn);
  w.tl.x = (float*)take(4 * (size_t)Tn);
  w.tl.chi2 = (float*)take(4 * (size_t)Tn);
  w.tl.par = (float*)take(4 * 5 * (size_t)Tn);
  w.tl.cov = (float*)take(4 * 15 * (size_t)Tn);
  w.tl.rowhit = (int32_t*)take(4 * (size_t)R * (size_t)Tn);
  w.tsel = (unsigned long long*)take(8 * (size_t)(Tn + 1));
  w.tscan = (unsigned long long*)take(8 * (size_t)(Tn + 1));
  w.kept_first = (int32_t*)take(4 * (size_t)Tn);
  w.kept_last = (int32_t*)take(4 * (size_t)Tn);
  w.owner_key = (unsigned long long*)take(8 * (size_t)Nn);
  w.owner_id = (uint32_t*)take(4 * (size_t)Nn);
  const size_t mgb = (int64_t)nb * MG_BINS < (1ll << 31) ? (size_t)nb * MG_BINS + 1 : 1;   // else: merger refused
  w.mg_start = (uint32_t*)take(4 * mgb);
  w.mg_fill = (uint32_t*)take(4 * mgb);
  w.mg_maxv = (uint32_t*)take(4 * (size_t)nb);
  w.mg_tiles = (uint32_t*)take(4 * (size_t)(ceilDiv((int64_t)mgb, SCAN_TILE) + 2));
  w.mg_list = (uint32_t*)take(4 * (size_t)Tn);
  w.mg_rec = (float4*)take(16 * (size_t)Tn);
  w.mg_ostart = (uint32_t*)take(4 * mgb);
  w.mg_ofill = (uint32_t*)take(4 * mgb);
  w.mg_order = (uint32_t*)take(4 * (size_t)Tn);
  const size_t rfb = (size_t)(Tn / RF_CHUNK + 1) * RF_BINS + 1;
  w.rf_hist = (uint32_t*)take(4 * rfb);
  w.rf_fill = (uint32_t*)take(4 * rfb);
  w.rf_order = (uint32_t*)take(4 * (size_t)Tn);
  w.mg_best_b = (int32_t*)take(4 * (size_t)Tn);
  w.mg_chi_b = (float*)take(4 * (size_t)Tn);
  w.mg_key_a = (unsigned long long*)take(8 * (size_t)Tn);
  w.fl_key = (unsigned long long*)take(8 * (size_t)Nn);
  w.fl_prot = (uint32_t*)take(4 * (size_t)ceilDiv(Nn, 32));
  w.mt_tiles = (uint32_t*)take(4 * (size_t)(ceilDiv(Tn + 1, SCAN_TILE) + 2));
  const size_t lgb = (int64_t)nb * 2 * LEG_BINS < (1ll << 31) ? (size_t)nb * 2 * LEG_BINS + 1 : 1;   // else: leg pairs refused
  w.lg_start = (uint32_t*)take(4 * lgb);
  w.lg_fill = (uint32_t*)take(4 * lgb);
  w.lg_maxv = (uint32_t*)take(4 * (size_t)nb * 2);
  w.lg_tiles = (uint32_t*)take(4 * (size_t)(ceilDiv((int64_t)lgb, SCAN_TILE) + 2));
  w.lg_list = (uint32_t*)take(4 * (size_t)Tn);
  w.lg_rec = (float4*)take(16 * (size_t)Tn);
  w.lg_best = (int32_t*)take(4 * (size_t)Tn);
  w.lg_chi = (float*)take(4 * (size_t)Tn);
  w.bytes = o;
  return w;
}

}  // namespace

extern "C" {

int tpcDefaultParams(tpcParams* p) {
  if (!p) return TPC_ERR_INVALID_ARG;
  p->area_y = 1.5f; p->area_z = 1.5f; p->link_dev2_max = 0.64f;
  p->err2_y = 0.01f; p->err2_z = 0.01f;
  p->init_var_s = 1.0f; p->init_var_t = 1.0f; p->init_var_q = 100.0f;
  p->turn_var_scale = 100.0f; p->max_sinphi = 0.98f;
  p->road_sigma = 4.0f; p->road_min = 0.3f; p->road_max = 2.0f;
  p->max_row_gap = 4; p->min_chain_hits = 3; p->min_tracklet_hits = 10; p->min_track_hits = 10;
  p->cell_min = 0.5f; p->cell_max = 8.0f; p->clusters_per_cell = 0.7f;
  p->validate_input = 0; p->force_wide_keys = 0;
  p->merge_max_row_gap = 40; p->merge_back_rows = 5; p->merge_chi2_max = 50.0f;
  p->tube_radius = 1.5f; p->inv_pt_protect = 20.0f; p->charge_trunc_bits = 4;
  p->leg_min_sinphi = 0.5f; p->leg_chi2_max = 50.0f; p->leg_max_sectors = 4; p->leg_max_row_diff = 12;
  p->leg_max_centre_dist = 10.0f; p->pos_bits = 6; p->tube_chi2_max = 0.0f;
  return TPC_OK;
}

int tpcCreate(tpcHandle** out, const tpcGeometry* g, const tpcParams* p, int cuda_device) {
  if (!out || !g || !p || !g->row_x) return TPC_ERR_INVALID_ARG;
  *out = nullptr;
  const int R = g->n_rows, S = g->n_sectors;
  if (R < 3 || R >= MAX_ROWS || S < 1 || S > 64) return TPC_ERR_INVALID_ARG;      // the hand-off records of the constructor carry the sector in 6 bits
  for (int r = 1; r < R; ++r)
    if (!(g->row_x[r] > g->row_x[r - 1])) return TPC_ERR_INVALID_ARG;
  if (!(g->z_max > g->z_min) || !(g->tan_half_sector > 0) || !(g->row_x[0] > 0)) return TPC_ERR_INVALID_ARG;
  if (!(p->cell_min > 0) || !(p->cell_max >= p->cell_min) || !(p->clusters_per_cell > 0)) return TPC_ERR_INVALID_ARG;
  if (p->min_chain_hits < 2 || p->max_row_gap < 0) return TPC_ERR_INVALID_ARG;
  if (p->merge_max_row_gap < 0 || p->merge_back_rows < 0) return TPC_ERR_INVALID_ARG;
  if (!(p->tube_chi2_max >= 0)) return TPC_ERR_INVALID_ARG;
  if (!(p->tube_radius >= 0) || p->charge_trunc_bits < 0 || p->charge_trunc_bits > 14) return TPC_ERR_INVALID_ARG;
  if (p->pos_bits < 0 || p->pos_bits > 15) return TPC_ERR_INVALID_ARG;
  if (p->leg_max_sectors < 0 || p->leg_max_sectors > LEG_MAX_SECTORS || p->leg_max_row_diff < 0) return TPC_ERR_INVALID_ARG;
  tpcHandle* h = new (std::nothrow) tpcHandle();
  if (!h) return TPC_ERR_OUT_OF_MEMORY;
  h->device = cuda_device;
  h->params = *p;
  DevParams& P = h->P;
  P.area_y = p->area_y; P.area_z = p->area_z; P.link_dev2_max = p->link_dev2_max;
  P.err2_y = p->err2_y; P.err2_z = p->err2_z; P.init_var_s = p->init_var_s; P.init_var_t = p->init_var_t;
  P.init_var_q = p->init_var_q; P.turn_var_scale = p->turn_var_scale; P.max_sinphi = p->max_sinphi;
  P.road_sigma = p->road_sigma; P.road_min = p->road_min; P.road_max = p->road_max;
  P.max_row_gap = p->max_row_gap; P.min_chain_hits = p->min_chain_hits; P.min_tracklet_hits = p->min_tracklet_hits;
  P.min_track_hits = p->min_track_hits; P.cell_min = p->cell_min; P.cell_max = p->cell_max;
  P.clusters_per_cell = p->clusters_per_cell;
  P.b = (float)(0.00299792458 * (double)g->bz_tesla);     // curvature constant, O4
  P.tan_half_sector = g->tan_half_sector; P.z_min = g->z_min; P.z_max = g->z_max;
  P.n_rows = R; P.n_sectors = S; P.n_buckets = R * S;
  P.max_cells_per_bucket = 1 << 24;
  h->row_x.assign(g->row_x, g->row_x + R);
  // R2: up(r) = first live row among r+1, r+2; dn(r) = first live row among r-1, r-2; none for dead rows
  std::vector<int16_t> up(R, -1), dn(R, -1);
  std::vector<uint8_t> dead(R, 0);
  for (int r = 0; r < R; ++r) dead[r] = (g->row_dead && g->row_dead[r]) ? 1 : 0;
  P.any_dead = 0;
  for (int r = 0; r < R; ++r) P.any_dead |= dead[r];
  for (int r = 0; r < R; ++r) {
    if (dead[r]) continue;
    for (int k = 1; k <= 2; ++k) if (r + k < R && !dead[r + k]) { up[r] = (int16_t)(r + k); break; }
    for (int k = 1; k <= 2; ++k) if (r - k >= 0 && !dead[r - k]) { dn[r] = (int16_t)(r - k); break; }
  }
  double bound = 0;
  const double Wz = (double)g->z_max - (double)g->z_min;
  for (int r = 0; r < R; ++r) {
    const double Wy = 2.0 * g->row_x[r] * g->tan_half_sector;
    bound += Wy * Wz / ((double)p->cell_max * p->cell_max) + (Wy + Wz) / p->cell_min + 2.0;
  }
  h->cells_per_bucket_bound = bound * S;
  cudaError_t e = cudaSetDevice(cuda_device);
  if (e != cudaSuccess) { delete h; return TPC_ERR_CUDA; }
  bool ok = cudaMalloc(&h->d_row_x, 4 * R) == cudaSuccess && cudaMalloc(&h->d_up, 2 * R) == cudaSuccess &&
            cudaMalloc(&h->d_dn, 2 * R) == cudaSuccess && cudaMalloc(&h->d_dead, R) == cudaSuccess &&
            cudaMalloc(&h->d_cnt, 8 * (CNT_COUNT + 1)) == cudaSuccess &&
            cudaMallocHost(&h->h_cnt, 8 * (CNT_COUNT + 1)) == cudaSuccess &&
            cudaEventCreate(&h->ev_done) == cudaSuccess;
  for (int i = 0; ok && i < 19; ++i) ok = cudaEventCreate(&h->ev_stage[i]) == cudaSuccess;
  ok = ok && cudaMemcpy(h->d_row_x, g->row_x, 4 * R, cudaMemcpyHostToDevice) == cudaSuccess &&
       cudaMemcpy(h->d_up, up.data(), 2 * R, cudaMemcpyHostToDevice) == cudaSuccess &&
       cudaMemcpy(h->d_dn, dn.data(), 2 * R, cudaMemcpyHostToDevice) == cudaSuccess &&
       cudaMemcpy(h->d_dead, dead.data(), R, cudaMemcpyHostToDevice) == cudaSuccess;
  if (!ok) { tpcDestroy(h); return TPC_ERR_CUDA; }
  {
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cuda_device);
    const void* pass[4] = {(const void*)constructUp, (const void*)constructDown<0, 0>, (const void*)constructDown<1, 0>,
                           (const void*)constructDown<0, 1>};
    for (int i = 0; i < 4; ++i) {
      int per_sm = 1;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pass[i], TC_THREADS, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
      h->tc_grid[i] = sms * per_sm;
    }
  }
  if (cudaFuncSetAttribute(gridBuild, cudaFuncAttributeMaxDynamicSharedMemorySize, h->gb_smem_bytes) != cudaSuccess) {
    cudaGetLastError();
    h->gb_smem_bytes = 4 * h->gb_smem_cells;      // the histogram alone: direct scatter
    if (cudaFuncSetAttribute(gridBuild, cudaFuncAttributeMaxDynamicSharedMemorySize, h->gb_smem_bytes) != cudaSuccess) {
      cudaGetLastError();
      h->gb_smem_cells = 10 * 1024;     // 40 KB needs no opt-in
      h->gb_smem_bytes = 4 * h->gb_smem_cells;
    }
  }
  memset(h->h_cnt, 0, 8 * (CNT_COUNT + 1));
  *out = h;
  return TPC_OK;
}

int tpcDestroy(tpcHandle* h) {
  if (!h) return TPC_ERR_INVALID_ARG;
  cudaSetDevice(h->device);
  cudaDeviceSynchronize();
  cudaFree(h->d_row_x); cudaFree(h->d_up); cudaFree(h->d_dn); cudaFree(h->d_dead); cudaFree(h->d_cnt);
  if (h->h_cnt) cudaFreeHost(h->h_cnt);
  if (h->ev_done) cudaEventDestroy(h->ev_done);
  for (int i = 0; i < 19; ++i) if (h->ev_stage[i]) cudaEventDestroy(h->ev_stage[i]);
  // the active state is freed below; the parked slots here, whatever part of them was initialised
  for (int k = 0; k < 3; ++k) {
    if (k == h->cur_slot) continue;
    tpcHandle::Slot& S = h->slots[k];
    if (S.d_cnt) cudaFree(S.d_cnt); if (S.h_cnt) cudaFreeHost(S.h_cnt); if (S.ev_done) cudaEventDestroy(S.ev_done);
    for (int i = 0; i < 16; ++i) if (S.pool[i]) cudaFree(S.pool[i]);
  }
  for (int k = 1; k < 3; ++k) {
    if (h->slots[k].stream) cudaStreamDestroy(h->slots[k].stream);
    if (h->slots[k].ev_begin) cudaEventDestroy(h->slots[k].ev_begin);
    if (h->slots[k].ev_kernels) cudaEventDestroy(h->slots[k].ev_kernels);
  }
  for (int i = 0; i < 16; ++i) if (h->pool[i]) cudaFree(h->pool[i]);
  delete h;
  return TPC_OK;
}

int tpcWorkspaceBytes(const tpcHandle* h, int64_t n_clusters, int64_t cap_tracklets, size_t* bytes) {
  if (!h || !bytes || n_clusters < 0 || n_clusters >= (1ll << 31) || cap_tracklets < 0 || cap_tracklets >= (1ll << 31))
    return TPC_ERR_INVALID_ARG;
  *bytes = layout(h, n_clusters, cap_tracklets, nullptr).bytes;
  return TPC_OK;
}

int tpcSetProfiling(tpcHandle* h, int on) {
  if (!h) return TPC_ERR_INVALID_ARG;
  h->profiling = on ? 1 : 0;
  return TPC_OK;
}

int tpcRun(tpcHandle* h, const tpcClusters* in, tpcTracks* out, int64_t cap_tracklets, void* workspace,
           size_t workspace_bytes, void* cuda_stream) {
  if (!h || !in || !out) return TPC_ERR_INVALID_ARG;
  const int64_t N = in->n_clusters, capT = cap_tracklets;
  if (N < 0 || N >= (1ll << 31) || capT < 0 || capT >= (1ll << 31) || !in->row_offset) return TPC_ERR_INVALID_ARG;
  if (N > 0 && (!in->y || !in->z)) return TPC_ERR_INVALID_ARG;
  if (out->cap_tracks < 0 || out->cap_track_clusters < 0 || out->cap_tracks >= (1ll << 31) ||
      out->cap_track_clusters >= (1ll << 32))
    return TPC_ERR_INVALID_ARG;
  if (!out->trk_cl_offset) return TPC_ERR_INVALID_ARG;
  if (out->cap_tracks > 0 && (!out->trk_tracklet || !out->trk_sector || !out->trk_first_row || !out->trk_last_row ||
                              !out->trk_ncl || !out->trk_x || !out->trk_par || !out->trk_cov || !out->trk_chi2))
    return TPC_ERR_INVALID_ARG;
  if (out->cap_track_clusters > 0 && !out->trk_cl_index) return TPC_ERR_INVALID_ARG;
  const int n_rf = (out->trk_rf_status != nullptr) + (out->trk_rf_x_in != nullptr) + (out->trk_rf_par_in != nullptr) +
                   (out->trk_rf_cov_in != nullptr) + (out->trk_rf_chi2 != nullptr) + (out->trk_rf_x_out != nullptr) +
                   (out->trk_rf_par_out != nullptr) + (out->trk_rf_cov_out != nullptr);
  if (n_rf != 0 && n_rf != 8) return TPC_ERR_INVALID_ARG;      // the refit outputs come all or none
  const int n_mg = (out->trk_mg_next != nullptr) + (out->trk_mg_prev != nullptr) + (out->trk_mg_head != nullptr) +
                   (out->trk_mg_chi2 != nullptr);
  if ((n_mg != 0 && n_mg != 4) || (n_mg == 4 && n_rf != 8)) return TPC_ERR_INVALID_ARG;   // the merger needs the refit
  if (n_mg == 4 && (int64_t)h->P.n_buckets * MG_BINS >= (1ll << 31)) return TPC_ERR_INVALID_ARG;   // bucket ids are 32-bit
  const int n_lg = (out->trk_leg_partner != nullptr) + (out->trk_leg_chi2 != nullptr);
  if ((n_lg != 0 && n_lg != 2) || (n_lg == 2 && n_rf != 8)) return TPC_ERR_INVALID_ARG;   // the leg pairs need the refit
  if (n_lg == 2 && (int64_t)h->P.n_buckets * 2 * LEG_BINS >= (1ll << 31)) return TPC_ERR_INVALID_ARG;   // bucket ids are 32-bit
  if (out->cl_qcode && N > 0 && !in->q) return TPC_ERR_INVALID_ARG;                      // the charge code needs the charges
  const int n_fl = (out->cl_flags != nullptr) + (out->cl_owner != nullptr);
  if ((n_fl != 0 && n_fl != 2) || (n_fl == 2 && n_rf != 8)) return TPC_ERR_INVALID_ARG;   // so do the cluster flags
  if ((out->cl_res_y != nullptr) != (out->cl_res_z != nullptr) || (out->cl_res_y && n_fl != 2)) return TPC_ERR_INVALID_ARG;
  if (out->cl_res_code && n_fl != 2) return TPC_ERR_INVALID_ARG;                         // the residual code rides on the flag pass
  const int n_mt = (out->trk_mt_id != nullptr) + (out->trk_mt_rank != nullptr) + (out->mt_cl_offset != nullptr) +
                   (out->mt_cl_index != nullptr);
  if ((n_mt != 0 && n_mt != 4) || (n_mt == 4 && (n_mg != 4 || n_lg != 2))) return TPC_ERR_INVALID_ARG;   // chains and leg pairs
  if (!workspace || ((uintptr_t)workspace % ALIGN) != 0) return TPC_ERR_INVALID_ARG;
  const Workspace w = layout(h, N, capT, (char*)workspace);
  if (workspace_bytes < w.bytes) return TPC_ERR_WORKSPACE_TOO_SMALL;
  TPC_CUDA(h, cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const DevParams& P = h->P;
  const int nb = P.n_buckets;
  const RowTables T{h->d_row_x, h->d_up, h->d_dn, h->d_dead};
  int64_t* cnt = h->d_cnt;
  const int wide = (h->params.force_wide_keys || capT >= (1ll << 24)) ? 1 : 0;
  int L = 0;
  auto stage = [&](int i) { if (h->profiling) cudaEventRecord(h->ev_stage[i], st); };
  const unsigned gN256 = (unsigned)ceilDiv(N, 256);
  const int64_t cc = capCells(h, N);

  stage(0);
  TPC_CUDA(h, cudaMemsetAsync(cnt, 0, 8 * (CNT_COUNT + 1), st)); ++L;
  // ---- a1 grid ----------------------------------------------------------------------------------
  gridSetup<<<1, 1024, 0, st>>>(in->row_offset, N, P, h->d_row_x, w.desc, w.chunk_base, NF_THREADS, cnt, cc); TPC_LAUNCHED("gridSetup");
  if (N > 0) {
    gridBuild<<<(unsigned)nb, GB_THREADS, (size_t)h->gb_smem_bytes, st>>>(in->row_offset, in->y, in->z, nb, w.desc, w.cell_start,
                                                                          w.rank, w.syz, w.s2o, cnt, h->params.validate_input,
                                                                          (uint32_t)h->gb_smem_cells, (uint32_t)h->gb_smem_bytes); TPC_LAUNCHED("gridBuild");
  }
  stage(1);
  // ---- a2 neighbour finder ------------------------------------------------------------------------
  if (N > 0) {
    // one CTA per chunk of NF_THREADS clusters of one bucket; the exact CTA count is on the device (chunk_base[nb])
    const int64_t max_chunks = ceilDiv(N, NF_THREADS) + nb;
    chunkFill<<<(unsigned)ceilDiv(max_chunks, 256), 256, 0, st>>>(w.chunk_base, nb, max_chunks, w.chunk_bucket, cnt); TPC_LAUNCHED("chunkFill");
    chunkRegions<<<(unsigned)ceilDiv(max_chunks * 32, 256), 256, 0, st>>>(w.chunk_base, w.chunk_bucket, P, T, w.desc, w.cell_start,
                                                                          w.syz, w.chunk_reg, cnt); TPC_LAUNCHED("chunkRegions");
    neighbourFinder<<<(unsigned)max_chunks, NF_THREADS, 0, st>>>(w.chunk_base, w.chunk_bucket, w.chunk_reg, P, T, w.desc, w.cell_start,
                                                                                    w.syz, w.s2o, w.lup, w.ldn, cnt); TPC_LAUNCHED("neighbourFinder");
  }
  stage(2);
  // ---- a3 cleaner + start hits --------------------------------------------------------------------
  const int64_t cpTiles = N > 0 ? ceilDiv(N, CP_TILE) : 0;
  uint32_t* cpTile = w.tiles32 + ceilDiv(cc + 1, SCAN_TILE) + 1;
  if (N > 0) {
    TPC_CUDA(h, cudaMemsetAsync(w.spos_by_orig, 0xFF, 4 * (size_t)N, st)); ++L;
    cleanLinks<<<gN256, 256, 0, st>>>(N, w.lup, w.ldn, w.s2o, w.cup, w.cdn, w.spos_by_orig, cnt); TPC_LAUNCHED("cleanLinks");
    startCount<<<(unsigned)cpTiles, CP_THREADS, 0, st>>>(N, w.spos_by_orig, cpTile); TPC_LAUNCHED("startCount");
  }
  scanArrayInPlace<uint32_t><<<1, 1024, 0, st>>>(cpTile, cpTiles, cnt + CNT_N_START); TPC_LAUNCHED("scanArrayInPlace<uint32_t>");
  if (N > 0 && capT > 0) {
    startWrite<<<(unsigned)cpTiles, CP_THREADS, 0, st>>>(N, w.spos_by_orig, cpTile, capT, w.start_orig, w.start_pos); TPC_LAUNCHED("startWrite");
  }
  stage(3);
  // ---- a4 tracklet constructor --------------------------------------------------------------------
  if (N > 0 && capT > 0) {
    const int64_t blocks = ceilDiv(capT, TC_THREADS);
    seedPrepare<<<(unsigned)ceilDiv(capT, 128), 128, 0, st>>>(in->row_offset, P, T, w.syz, w.cup, w.start_pos, w.work_list,
                                                              w.tl, cnt); TPC_LAUNCHED("seedPrepare");
    constructUp<<<(unsigned)std::min<int64_t>(blocks, h->tc_grid[0]), TC_THREADS, 0, st>>>(
        P, T, w.desc, w.cell_start, w.syz, w.s2o, w.cup, w.work_list, w.turn_list, w.tl, cnt); TPC_LAUNCHED("constructUp");
    gapListBuild<<<(unsigned)ceilDiv(capT, 1024), 1024, 0, st>>>(w.turn_list, w.gap_idx, cnt); TPC_LAUNCHED("gapListBuild");
    constructDown<0, 0><<<(unsigned)std::min<int64_t>(blocks, h->tc_grid[1]), TC_THREADS, 0, st>>>(
        P, T, w.desc, w.cell_start, w.syz, w.s2o, w.turn_list, w.gap_idx, w.down_list, w.tl, cnt); TPC_LAUNCHED("constructDown<0, 0>");
    constructDown<0, 1><<<(unsigned)std::min<int64_t>(blocks, h->tc_grid[3]), TC_THREADS, 0, st>>>(
        P, T, w.desc, w.cell_start, w.syz, w.s2o, w.turn_list, w.gap_idx, w.down_list, w.tl, cnt); TPC_LAUNCHED("constructDown<0, 1>");
    constructDown<1, 0><<<(unsigned)std::min<int64_t>(blocks, h->tc_grid[2]), TC_THREADS, 0, st>>>(
        P, T, w.desc, w.cell_start, w.syz, w.s2o, w.turn_list, w.gap_idx, w.down_list, w.tl, cnt); TPC_LAUNCHED("constructDown<1, 0>");
  }
  stage(4);
  // optional per-stage export of the tracklets: before the selector, which compacts the row-hit slices in place
  if (N > 0 && capT > 0 && (out->start_hits || out->tl_status || out->tl_nhits || out->tl_first_row || out->tl_last_row ||
                            out->tl_rowhit || out->tl_x || out->tl_par || out->tl_cov || out->tl_chi2)) {
    const TrackletOut xo{out->start_hits, out->tl_status, out->tl_nhits, out->tl_first_row, out->tl_last_row,
                         out->tl_rowhit, out->tl_x, out->tl_par, out->tl_cov, out->tl_chi2};
    exportTracklets<<<(unsigned)ceilDiv(capT, 128), 128, 0, st>>>(w.tl, w.start_orig, w.s2o, P.n_rows, xo, cnt); TPC_LAUNCHED("exportTracklets");
  }
  // ---- a5 selector ----------------------------------------------------------------------------------
  const TrackOut to{out->cap_tracks, out->cap_track_clusters, out->trk_tracklet, out->trk_sector, out->trk_first_row,
                    out->trk_last_row, out->trk_ncl, out->trk_x, out->trk_par, out->trk_cov, out->trk_chi2,
                    out->trk_cl_offset, out->trk_cl_index};
  unsigned long long* sel_total = (unsigned long long*)(cnt + CNT_COUNT);
  if (N > 0 && capT > 0) {
    const unsigned gT = (unsigned)ceilDiv(capT, 128);
    TPC_CUDA(h, cudaMemsetAsync(w.owner_key, 0, 8 * (size_t)N, st)); ++L;
    selectClaim<<<gT, 128, 0, st>>>(w.tl, w.owner_key, wide, cnt); TPC_LAUNCHED("selectClaim");
    if (wide) {
      TPC_CUDA(h, cudaMemsetAsync(w.owner_id, 0xFF, 4 * (size_t)N, st)); ++L;
      selectClaimId<<<gT, 128, 0, st>>>(w.tl, w.owner_key, w.owner_id, cnt); TPC_LAUNCHED("selectClaimId");
    }
    selectCount<<<gT, 128, 0, st>>>(w.tl, w.owner_key, w.owner_id, wide, P.min_track_hits, w.tsel, w.kept_first,
                                    w.kept_last, cnt); TPC_LAUNCHED("selectCount");
    const unsigned tiles = (unsigned)ceilDiv(capT, SCAN_TILE);
    scanTileSums<unsigned long long><<<tiles, SCAN_THREADS, 0, st>>>(w.tsel, cnt + CNT_N_START, capT, w.tiles64); TPC_LAUNCHED("scanTileSums<unsigned long long>");
    scanTileOffsets<unsigned long long><<<1, 1024, 0, st>>>(w.tiles64, cnt + CNT_N_START, capT, sel_total); TPC_LAUNCHED("scanTileOffsets<unsigned long long>");
    scanApply<unsigned long long><<<tiles, SCAN_THREADS, 0, st>>>(w.tsel, w.tscan, cnt + CNT_N_START, capT, w.tiles64); TPC_LAUNCHED("scanApply<unsigned long long>");
    selectEmit<<<gT, 128, 0, st>>>(w.tl, w.owner_key, w.owner_id, wide, w.tsel, w.tscan, w.kept_first, w.kept_last,
                                   w.s2o, to, cnt); TPC_LAUNCHED("selectEmit");
  }
  finalize<<<1, 32, 0, st>>>(sel_total, to, capT, cnt); TPC_LAUNCHED("finalize");
  stage(5);
  // ---- a6 optional refit of the selected tracks (O6) ------------------------------------------------
  stage(7);
  if (n_rf == 8 && N > 0 && out->cap_tracks > 0) {
    const RefitOut rf{out->trk_rf_status, out->trk_rf_x_in, out->trk_rf_par_in, out->trk_rf_cov_in, out->trk_rf_chi2,
                      out->trk_rf_x_out, out->trk_rf_par_out, out->trk_rf_cov_out};
    const int64_t nk = std::min<int64_t>(out->cap_tracks, capT);
    const size_t rfb = (size_t)(nk / RF_CHUNK + 1) * RF_BINS + 1;
    TPC_CUDA(h, cudaMemsetAsync(w.rf_hist, 0, 4 * rfb, st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(w.rf_fill, 0, 4 * rfb, st)); ++L;
    refitCount<<<(unsigned)ceilDiv(nk, 256), 256, 0, st>>>(to, w.rf_hist, cnt); TPC_LAUNCHED("refitCount");
    scanArrayInPlace<uint32_t><<<1, 1024, 0, st>>>(w.rf_hist, (int64_t)rfb, nullptr); TPC_LAUNCHED("scanArrayInPlace<uint32_t>");
    refitFill<<<(unsigned)ceilDiv(nk, 256), 256, 0, st>>>(to, w.rf_hist, w.rf_fill, w.rf_order, cnt); TPC_LAUNCHED("refitFill");
    refitTracks<<<(unsigned)ceilDiv(nk, 128), 128, 0, st>>>(in->row_offset, w.rf_order, in->y, in->z, P, T, to, rf, cnt); TPC_LAUNCHED("refitTracks");
  }
  stage(8);
  // ---- a7 optional links between track segments (O7) -------------------------------------------------
  stage(9);
  if (n_mg == 4 && N > 0 && out->cap_tracks > 0) {
    const int64_t nk = std::min<int64_t>(out->cap_tracks, capT);     // tracks <= tracklets <= capT: the lists fit
    const MergeIn mi{out->cap_tracks, out->trk_rf_status, out->trk_sector, out->trk_first_row, out->trk_last_row,
                     out->trk_rf_x_in, out->trk_rf_par_in, out->trk_rf_cov_in, out->trk_rf_x_out, out->trk_rf_par_out,
                     out->trk_rf_cov_out};
    const MergeOut mo{out->trk_mg_next, out->trk_mg_prev, out->trk_mg_head, out->trk_mg_chi2};
    const MergeParams mp{h->params.merge_max_row_gap, h->params.merge_back_rows, h->params.merge_chi2_max,
                         (float)cos(0.3490658503988659), (float)sin(0.3490658503988659)};
    const unsigned gK = (unsigned)ceilDiv(nk, 256);
    const size_t mgb = (size_t)nb * MG_BINS + 1;
    TPC_CUDA(h, cudaMemsetAsync(w.mg_start, 0, 4 * mgb, st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(w.mg_fill, 0, 4 * mgb, st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(w.mg_ostart, 0, 4 * mgb, st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(w.mg_ofill, 0, 4 * mgb, st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(w.mg_maxv, 0, 4 * (size_t)nb, st)); ++L;
    mergeCount<<<gK, 256, 0, st>>>(mi, mo, P, T, w.mg_start, w.mg_ostart, w.mg_maxv, w.mg_best_b, w.mg_key_a, cnt); TPC_LAUNCHED("mergeCount");
    {   // exclusive scan of the bucket counts; the closing sentinel lands on the last (spare) entry
      const int64_t nscan = (int64_t)mgb - 1;
      const unsigned tiles = (unsigned)ceilDiv(nscan, SCAN_TILE);
      scanTileSums<uint32_t><<<tiles, SCAN_THREADS, 0, st>>>(w.mg_start, cnt + CNT_INF, nscan, w.mg_tiles); TPC_LAUNCHED("scanTileSums<uint32_t>");
      scanTileOffsets<uint32_t><<<1, 1024, 0, st>>>(w.mg_tiles, cnt + CNT_INF, nscan, nullptr); TPC_LAUNCHED("scanTileOffsets<uint32_t>");
      scanApply<uint32_t><<<tiles, SCAN_THREADS, 0, st>>>(w.mg_start, w.mg_start, cnt + CNT_INF, nscan, w.mg_tiles); TPC_LAUNCHED("scanApply<uint32_t>");
      scanTileSums<uint32_t><<<tiles, SCAN_THREADS, 0, st>>>(w.mg_ostart, cnt + CNT_INF, nscan, w.mg_tiles); TPC_LAUNCHED("scanTileSums<uint32_t>");
      scanTileOffsets<uint32_t><<<1, 1024, 0, st>>>(w.mg_tiles, cnt + CNT_INF, nscan, nullptr); TPC_LAUNCHED("scanTileOffsets<uint32_t>");
      scanApply<uint32_t><<<tiles, SCAN_THREADS, 0, st>>>(w.mg_ostart, w.mg_ostart, cnt + CNT_INF, nscan, w.mg_tiles); TPC_LAUNCHED("scanApply<uint32_t>");
    }
    mergeFill<<<gK, 256, 0, st>>>(mi, P, T, w.mg_start, w.mg_fill, w.mg_list, w.mg_rec, w.mg_ostart, w.mg_ofill, w.mg_order, cnt); TPC_LAUNCHED("mergeFill");
    mergeMatch<<<(unsigned)ceilDiv(nk, 128), 128, 0, st>>>(mi, P, T, mp, w.mg_start, w.mg_maxv, w.mg_list, w.mg_rec, w.mg_ostart, w.mg_order, w.mg_best_b,
                                                         w.mg_chi_b, w.mg_key_a, cnt); TPC_LAUNCHED("mergeMatch");
    mergeLink<<<gK, 256, 0, st>>>(mi, mo, w.mg_best_b, w.mg_chi_b, w.mg_key_a, cnt); TPC_LAUNCHED("mergeLink");
    mergeHead<<<gK, 256, 0, st>>>(mi, mo, cnt); TPC_LAUNCHED("mergeHead");
  }
  stage(10);
  // ---- a10 optional pairs of looper legs (O10) -------------------------------------------------------
  stage(15);
  if (n_lg == 2 && N > 0 && out->cap_tracks > 0) {
    const int64_t nk = std::min<int64_t>(out->cap_tracks, capT);
    const LegIn li{out->cap_tracks, out->trk_rf_status, out->trk_sector, out->trk_last_row, out->trk_rf_x_out,
                   out->trk_rf_par_out, out->trk_rf_cov_out};
    const LegOut lo{out->trk_leg_partner, out->trk_leg_chi2};
    LegParams lp{};
    lp.min_sinphi = h->params.leg_min_sinphi; lp.chi2_max = h->params.leg_chi2_max;
    lp.max_sectors = h->params.leg_max_sectors; lp.max_row_diff = h->params.leg_max_row_diff;
    lp.max_centre_dist = h->params.leg_max_centre_dist;
    for (int d = -LEG_MAX_SECTORS; d <= LEG_MAX_SECTORS; ++d)
      for (int sg = -1; sg <= 1; sg += 2) {
        if (d * sg < 0) continue;                  // a moves towards b's sector
        const double a10 = 0.17453292519943295, a90 = 1.5707963267948966;
        const double alpha = (double)d * a10 + (double)sg * a90;
        const int i = d + LEG_MAX_SECTORS + (sg > 0 ? 1 : 0);
        lp.ca[i] = (float)cos(alpha); lp.sa[i] = (float)sin(alpha);
        lp.cb[i] = (float)cos(-alpha); lp.sb[i] = (float)sin(-alpha);
      }
    for (int d = -LEG_MAX_SECTORS; d <= LEG_MAX_SECTORS; ++d) {
      const double a10 = 0.17453292519943295;
      lp.cd[d + LEG_MAX_SECTORS] = (float)cos((double)d * (2.0 * a10)); lp.sd[d + LEG_MAX_SECTORS] = (float)sin((double)d * (2.0 * a10));
    }
    const unsigned gK = (unsigned)ceilDiv(nk, 256);
    const size_t lgb = (size_t)nb * 2 * LEG_BINS + 1;
    TPC_CUDA(h, cudaMemsetAsync(w.lg_start, 0, 4 * lgb, st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(w.lg_fill, 0, 4 * lgb, st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(w.lg_maxv, 0, 4 * (size_t)nb * 2, st)); ++L;
    legCount<<<gK, 256, 0, st>>>(li, lo, P, lp, w.lg_start, w.lg_maxv, w.lg_best, cnt); TPC_LAUNCHED("legCount");
    {   // exclusive scan of the bucket counts; the closing sentinel lands on the last (spare) entry
      const int64_t nscan = (int64_t)lgb - 1;
      const unsigned tiles = (unsigned)ceilDiv(nscan, SCAN_TILE);
      scanTileSums<uint32_t><<<tiles, SCAN_THREADS, 0, st>>>(w.lg_start, cnt + CNT_INF, nscan, w.lg_tiles); TPC_LAUNCHED("scanTileSums<uint32_t>");
      scanTileOffsets<uint32_t><<<1, 1024, 0, st>>>(w.lg_tiles, cnt + CNT_INF, nscan, nullptr); TPC_LAUNCHED("scanTileOffsets<uint32_t>");
      scanApply<uint32_t><<<tiles, SCAN_THREADS, 0, st>>>(w.lg_start, w.lg_start, cnt + CNT_INF, nscan, w.lg_tiles); TPC_LAUNCHED("scanApply<uint32_t>");
    }
    legFill<<<gK, 256, 0, st>>>(li, P, lp, w.lg_start, w.lg_fill, w.lg_list, w.lg_rec, cnt); TPC_LAUNCHED("legFill");
    legMatch<<<(unsigned)ceilDiv(nk, 128), 128, 0, st>>>(li, P, lp, w.lg_start, w.lg_maxv, w.lg_list, w.lg_rec, w.lg_best,
                                                         w.lg_chi, cnt); TPC_LAUNCHED("legMatch");
    legLink<<<gK, 256, 0, st>>>(li, lo, w.lg_best, w.lg_chi, cnt); TPC_LAUNCHED("legLink");
  }
  stage(16);
  // ---- a11 optional merged tracks and leg labels (O12) ------------------------------------------------
  stage(17);
  if (n_mt == 4 && N > 0 && out->cap_tracks > 0) {
    const int64_t nk = std::min<int64_t>(out->cap_tracks, capT);
    const MergedIn mi{out->cap_tracks, out->trk_mg_next, out->trk_mg_head, out->trk_leg_partner, out->trk_cl_offset,
                      out->trk_cl_index, in->z};
    const MergedOut mo{out->trk_mt_id, out->trk_mt_rank, out->mt_cl_offset, out->mt_cl_index};
    mergedLabel<<<(unsigned)ceilDiv(nk + 1, 256), 256, 0, st>>>(mi, mo, cnt); TPC_LAUNCHED("mergedLabel");
    // exclusive scan of the lengths in place: n_tracks entries and the closing one (the scan writes out[n] itself)
    const unsigned tiles = (unsigned)ceilDiv(nk + 1, SCAN_TILE);
    scanTileSums<uint32_t><<<tiles, SCAN_THREADS, 0, st>>>(out->mt_cl_offset, cnt + CNT_N_TRACKS, nk, w.mt_tiles); TPC_LAUNCHED("scanTileSums<uint32_t>");
    scanTileOffsets<uint32_t><<<1, 1024, 0, st>>>(w.mt_tiles, cnt + CNT_N_TRACKS, nk, nullptr); TPC_LAUNCHED("scanTileOffsets<uint32_t>");
    scanApply<uint32_t><<<tiles, SCAN_THREADS, 0, st>>>(out->mt_cl_offset, out->mt_cl_offset, cnt + CNT_N_TRACKS, nk, w.mt_tiles); TPC_LAUNCHED("scanApply<uint32_t>");
    mergedFill<<<(unsigned)ceilDiv(nk, 128), 128, 0, st>>>(mi, mo, out->cap_track_clusters, cnt); TPC_LAUNCHED("mergedFill");
  }
  stage(18);
  // ---- a8 optional per-cluster flags (O8) ------------------------------------------------------------
  stage(11);
  if (n_fl == 2 && N > 0) {
    TPC_CUDA(h, cudaMemsetAsync(w.fl_key, 0xFF, 8 * (size_t)N, st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(w.fl_prot, 0, 4 * (size_t)ceilDiv(N, 32), st)); ++L;
    TPC_CUDA(h, cudaMemsetAsync(out->cl_flags, 0, (size_t)N, st)); ++L;
    if (out->cl_res_code) { TPC_CUDA(h, cudaMemsetAsync(out->cl_res_code, 0, 4 * (size_t)N, st)); ++L; }
    if (out->cl_res_y) {
      TPC_CUDA(h, cudaMemsetAsync(out->cl_res_y, 0, 4 * (size_t)N, st)); ++L;
      TPC_CUDA(h, cudaMemsetAsync(out->cl_res_z, 0, 4 * (size_t)N, st)); ++L;
    }
    if (out->cap_tracks > 0 && out->cap_track_clusters > 0) {
      const FlagIn fi{out->cap_tracks, out->trk_rf_status, out->trk_sector, out->trk_first_row, out->trk_last_row,
                      out->trk_rf_x_in, out->trk_rf_par_in, out->trk_rf_cov_in, out->trk_cl_offset, out->trk_cl_index};
      const int64_t nk = std::min<int64_t>(out->cap_tracks, capT);
      // the walking states of the attached clusters, one float2 per track-cluster entry: the selector's owner keys
      // (8 bytes per cluster, dead since selectEmit) are the buffer
      float2* walk_yz = (out->cl_res_y || out->cl_res_code) ? reinterpret_cast<float2*>(w.owner_key) : nullptr;
      const int64_t n_ent = std::min<int64_t>(out->cap_track_clusters, N);
      if (walk_yz) { TPC_CUDA(h, cudaMemsetAsync(walk_yz, 0xFF, 8 * (size_t)n_ent, st)); ++L; }
      flagAttach<<<(unsigned)ceilDiv(std::min<int64_t>(out->cap_track_clusters, N), 256), 256, 0, st>>>(out->trk_cl_index,
                                                                                                       out->cl_flags, cnt); TPC_LAUNCHED("flagAttach");
      const unsigned gB = (unsigned)ceilDiv(nk * FLAG_GROUP, 128);
      const int32_t* rk = n_mt == 4 ? out->trk_mt_rank : nullptr;
      if (h->params.tube_chi2_max > 0.0f)
        flagBid<1><<<gB, 128, 0, st>>>(fi, in->row_offset, P, T, h->params.tube_radius, h->params.tube_chi2_max,
                                       h->params.inv_pt_protect, w.desc, w.cell_start, w.syz, w.s2o, w.fl_key, w.fl_prot, rk,
                                       walk_yz, cnt);
      else
        flagBid<0><<<gB, 128, 0, st>>>(fi, in->row_offset, P, T, h->params.tube_radius, 0.0f, h->params.inv_pt_protect, w.desc,
                                       w.cell_start, w.syz, w.s2o, w.fl_key, w.fl_prot, rk, walk_yz, cnt);
      TPC_LAUNCHED("flagBid");
      if (walk_yz) {
        flagResiduals<<<(unsigned)ceilDiv(n_ent, 256), 256, 0, st>>>(out->trk_cl_index, walk_yz, in->y, in->z, out->cl_res_y,
                                                                    out->cl_res_z, out->cl_res_code, h->params.pos_bits, cnt); TPC_LAUNCHED("flagResiduals");
      }
    }
    flagFinish<<<gN256, 256, 0, st>>>(N, w.fl_key, w.fl_prot, out->cl_flags, out->cl_owner, cnt); TPC_LAUNCHED("flagFinish");
  }
  stage(12);
  // ---- a9 optional dynamic-precision charge code (O9) ------------------------------------------------
  stage(13);
  if (out->cl_qcode && N > 0) {
    packCharge<<<(unsigned)ceilDiv(ceilDiv(N, 8), 256), 256, 0, st>>>(N, in->q, h->params.charge_trunc_bits, out->cl_qcode); TPC_LAUNCHED("packCharge");
  }
  if (out->cl_pos_code && N > 0) {    // O11 of the absolute positions
    packPositions<<<(unsigned)ceilDiv(ceilDiv(N, 4), 256), 256, 0, st>>>(N, in->y, in->z, h->params.pos_bits, out->cl_pos_code); TPC_LAUNCHED("packPositions");
  }
  stage(14);
  // ---- optional per-stage exports -----------------------------------------------------------------
  if (N > 0 && (out->link_up_raw || out->link_dn_raw || out->link_up || out->link_dn)) {
    exportLinks<<<gN256, 256, 0, st>>>(N, w.s2o, w.lup, w.ldn, w.cup, w.cdn, out->link_up_raw, out->link_dn_raw,
                                       out->link_up, out->link_dn, cnt); TPC_LAUNCHED("exportLinks");
  }
  stage(6);
  TPC_CUDA(h, cudaGetLastError());
  TPC_CUDA(h, cudaMemcpyAsync(h->h_cnt, cnt, 8 * (CNT_COUNT + 1), cudaMemcpyDeviceToHost, st));
  TPC_CUDA(h, cudaEventRecord(h->ev_done, st));
  h->launches = L;
  h->pending = true;
  h->last_n = N;
  return TPC_OK;
}

int tpcGetRunStatus(tpcHandle* h, tpcRunStatus* out) {
  if (!h || !out) return TPC_ERR_INVALID_ARG;
  if (!h->pending) return TPC_ERR_INVALID_ARG;
  TPC_CUDA(h, cudaEventSynchronize(h->ev_done));
  memset(out, 0, sizeof(*out));
  const int64_t* c = h->h_cnt;
  out->status = (int32_t)c[CNT_ERROR];
  out->kernel_launches = h->launches;
  out->n_clusters = h->last_n;
  out->n_start_hits = c[CNT_N_START];
  out->n_tracklets = c[CNT_N_TRACKLETS];
  out->n_tracklet_hits = c[CNT_N_TL_HITS];
  out->n_tracks = c[CNT_N_TRACKS];
  out->n_track_clusters = c[CNT_N_TRK_CL];
  out->n_cells = c[CNT_N_CELLS];
  if (h->profiling) {
    for (int i = 0; i < 6; ++i) {
      float ms = 0;
      if (cudaEventElapsedTime(&ms, h->ev_stage[i], h->ev_stage[i + 1]) == cudaSuccess) out->stage_ms[i] = ms;
    }
    float ms = 0;
    if (cudaEventElapsedTime(&ms, h->ev_stage[0], h->ev_stage[6]) == cudaSuccess) out->stage_ms[6] = ms;
    if (cudaEventElapsedTime(&ms, h->ev_stage[7], h->ev_stage[8]) == cudaSuccess) out->stage_ms[7] = ms;
    if (cudaEventElapsedTime(&ms, h->ev_stage[9], h->ev_stage[10]) == cudaSuccess) out->merge_ms = ms;
    if (cudaEventElapsedTime(&ms, h->ev_stage[11], h->ev_stage[12]) == cudaSuccess) out->flags_ms = ms;
    if (cudaEventElapsedTime(&ms, h->ev_stage[13], h->ev_stage[14]) == cudaSuccess) out->pack_ms = ms;
    if (cudaEventElapsedTime(&ms, h->ev_stage[15], h->ev_stage[16]) == cudaSuccess) out->legs_ms = ms;
    if (cudaEventElapsedTime(&ms, h->ev_stage[17], h->ev_stage[18]) == cudaSuccess) out->merged_ms = ms;
  }
  return TPC_OK;
}

const char* tpcErrorString(int code) {
  switch (code) {
    case TPC_OK: return "ok";
    case TPC_ERR_INVALID_ARG: return "invalid argument";
    case TPC_ERR_UNSORTED_OFFSETS: return "row_offset is not a monotone CSR offset array ending at n_clusters";
    case TPC_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case TPC_ERR_CAPACITY: return "output capacity exceeded (outputs truncated; see tpcRunStatus for required sizes)";
    case TPC_ERR_CUDA: return "CUDA runtime error";
    case TPC_ERR_NONFINITE_INPUT: return "non-finite cluster coordinate";
    case TPC_ERR_OUT_OF_MEMORY: return "out of host memory";
    case TPC_ERR_NOALLOC_LIMIT: return "input larger than the static scratch of the allocation-free entry point (TPC_NOALLOC_MAX_CLUSTERS)";
    default: return "unknown error";
  }
}

const char* tpcLastCudaError(const tpcHandle* h) { return h ? h->cuda_msg : ""; }

int tpcSelfTestDivision(tpcHandle* h, int64_t n_threads, uint64_t seed, int64_t* n_tested, int64_t* n_mismatches) {
  if (!h || n_threads < 1 || n_threads > (1ll << 34) || !n_tested || !n_mismatches) return TPC_ERR_INVALID_ARG;
  TPC_CUDA(h, cudaSetDevice(h->device));
  unsigned long long* d = nullptr;
  TPC_CUDA(h, cudaMalloc(&d, 16));
  cudaError_t e = cudaMemset(d, 0, 16);
  if (e == cudaSuccess) {
    divisionSelfTest<<<(unsigned)ceilDiv(n_threads, 256), 256>>>((uint64_t)n_threads, seed, d, d + 1);
    e = cudaGetLastError();
  }
  unsigned long long r[2] = {0, 0};
  if (e == cudaSuccess) e = cudaMemcpy(r, d, 16, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return cudaFail(h, e, "tpcSelfTestDivision");
  *n_mismatches = (int64_t)r[0]; *n_tested = (int64_t)r[1];
  return TPC_OK;
}

}  // extern "C"

// ---- host-buffer convenience path ---------------------------------------------------------------------------
namespace {
int poolGet(tpcHandle* h, int idx, size_t bytes, void** p) {
  if (bytes == 0) bytes = ALIGN;
  if (h->pool_bytes[idx] < bytes) {
    if (h->pool[idx]) cudaFree(h->pool[idx]);
    h->pool[idx] = nullptr; h->pool_bytes[idx] = 0;
    const size_t want = bytes + bytes / 8;   // head-room so that slowly growing inputs do not reallocate every call
    TPC_CUDA(h, cudaMalloc(&h->pool[idx], want));
    h->pool_bytes[idx] = want;
  }
  *p = h->pool[idx];
  return TPC_OK;
}
}  // namespace

extern "C" int tpcRunHost(tpcHandle* h, int64_t N, const uint32_t* row_offset, const float* y, const float* z,
                          tpcTracks* oh, tpcRunStatus* status, void* cuda_stream) {
  if (!h || !row_offset || !oh || !status || N < 0 || N >= (1ll << 31) || (N > 0 && (!y || !z))) return TPC_ERR_INVALID_ARG;
  if (oh->link_up_raw || oh->link_dn_raw || oh->link_up || oh->link_dn || oh->start_hits || oh->tl_status || oh->tl_nhits ||
      oh->tl_first_row || oh->tl_last_row || oh->tl_rowhit || oh->tl_x || oh->tl_par || oh->tl_cov || oh->tl_chi2 ||
      oh->trk_rf_status || oh->trk_rf_x_in || oh->trk_rf_par_in || oh->trk_rf_cov_in || oh->trk_rf_chi2 || oh->trk_rf_x_out ||
      oh->trk_rf_par_out || oh->trk_rf_cov_out || oh->trk_mg_next || oh->trk_mg_prev || oh->trk_mg_head || oh->trk_mg_chi2 ||
      oh->trk_leg_partner || oh->trk_leg_chi2 || oh->cl_flags || oh->cl_owner || oh->cl_qcode || oh->cl_res_y || oh->cl_res_z || oh->cl_pos_code || oh->cl_res_code ||
      oh->trk_mt_id || oh->trk_mt_rank || oh->mt_cl_offset || oh->mt_cl_index)
    return TPC_ERR_INVALID_ARG;
  if (!oh->trk_cl_offset || oh->cap_tracks < 0 || oh->cap_track_clusters < 0) return TPC_ERR_INVALID_ARG;
  TPC_CUDA(h, cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int nb = h->P.n_buckets;
  int64_t capT = std::max<int64_t>(std::max<int64_t>(4096, N / 8), h->hint_T);
  int64_t capK = std::max<int64_t>(std::max<int64_t>(4096, N / 64), h->hint_K);
  int64_t capC = std::max<int64_t>(std::max<int64_t>(N / 2, 1), h->hint_C);
  void *d_off, *d_y, *d_z;
  int rc;
  if ((rc = poolGet(h, 0, 4 * (size_t)(nb + 1), &d_off)) || (rc = poolGet(h, 1, 4 * (size_t)N, &d_y)) ||
      (rc = poolGet(h, 2, 4 * (size_t)N, &d_z)))
    return rc;
  TPC_CUDA(h, cudaMemcpyAsync(d_off, row_offset, 4 * (size_t)(nb + 1), cudaMemcpyHostToDevice, st));
  if (N > 0) {
    TPC_CUDA(h, cudaMemcpyAsync(d_y, y, 4 * (size_t)N, cudaMemcpyHostToDevice, st));
    TPC_CUDA(h, cudaMemcpyAsync(d_z, z, 4 * (size_t)N, cudaMemcpyHostToDevice, st));
  }
  tpcTracks od{};
  for (int attempt = 0;; ++attempt) {
    size_t wsb = 0;
    if ((rc = tpcWorkspaceBytes(h, N, capT, &wsb))) return rc;
    void* ws;
    if ((rc = poolGet(h, 3, wsb, &ws))) return rc;
    void* p[11];
    const size_t K = (size_t)capK;
    const size_t sz[11] = {4 * K, 4 * K, 4 * K, 4 * K, 4 * K, 4 * K, 20 * K, 60 * K, 4 * K, 4 * (K + 1), 4 * (size_t)capC};
    for (int i = 0; i < 11; ++i)
      if ((rc = poolGet(h, 4 + i, sz[i], &p[i]))) return rc;
    od = tpcTracks{};
    od.cap_tracks = capK; od.cap_track_clusters = capC;
    od.trk_tracklet = (int32_t*)p[0]; od.trk_sector = (int32_t*)p[1]; od.trk_first_row = (int32_t*)p[2];
    od.trk_last_row = (int32_t*)p[3]; od.trk_ncl = (int32_t*)p[4]; od.trk_x = (float*)p[5]; od.trk_par = (float*)p[6];
    od.trk_cov = (float*)p[7]; od.trk_chi2 = (float*)p[8]; od.trk_cl_offset = (uint32_t*)p[9];
    od.trk_cl_index = (uint32_t*)p[10];
    const tpcClusters in{N, (const uint32_t*)d_off, nullptr, (const float*)d_y, (const float*)d_z, nullptr};
    if ((rc = tpcRun(h, &in, &od, capT, ws, h->pool_bytes[3], st))) return rc;
    if ((rc = tpcGetRunStatus(h, status))) return rc;
    if (status->status != TPC_ERR_CAPACITY || attempt >= 2) break;
    capT = std::max(capT, status->n_start_hits + status->n_start_hits / 16);
    capK = std::max(capK, status->n_tracks + status->n_tracks / 16);
    capC = std::max(capC, status->n_track_clusters + status->n_track_clusters / 16);
  }
  // the next call on similar data gets it right the first time
  h->hint_T = std::max(h->hint_T, status->n_start_hits + status->n_start_hits / 16);
  h->hint_K = std::max(h->hint_K, status->n_tracks + status->n_tracks / 16);
  h->hint_C = std::max(h->hint_C, status->n_track_clusters + status->n_track_clusters / 16);
  if (status->status != TPC_OK) return TPC_OK;   // data-dependent error: reported through *status
  const int64_t nt = std::min<int64_t>(status->n_tracks, oh->cap_tracks);
  const int64_t nc = status->n_track_clusters;
  if (status->n_tracks > oh->cap_tracks || nc > oh->cap_track_clusters) status->status = TPC_ERR_CAPACITY;
  auto back = [&](void* dst, const void* src, size_t bytes) {
    return (dst && bytes) ? cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st) : cudaSuccess;
  };
  const size_t n4 = 4 * (size_t)nt;
  TPC_CUDA(h, back(oh->trk_tracklet, od.trk_tracklet, n4));
  TPC_CUDA(h, back(oh->trk_sector, od.trk_sector, n4));
  TPC_CUDA(h, back(oh->trk_first_row, od.trk_first_row, n4));
  TPC_CUDA(h, back(oh->trk_last_row, od.trk_last_row, n4));
  TPC_CUDA(h, back(oh->trk_ncl, od.trk_ncl, n4));
  TPC_CUDA(h, back(oh->trk_x, od.trk_x, n4));
  TPC_CUDA(h, back(oh->trk_chi2, od.trk_chi2, n4));
  if (nt > 0 && oh->trk_par)
    TPC_CUDA(h, cudaMemcpy2DAsync(oh->trk_par, 4 * (size_t)oh->cap_tracks, od.trk_par, 4 * (size_t)od.cap_tracks, n4, 5,
                                  cudaMemcpyDeviceToHost, st));
  if (nt > 0 && oh->trk_cov)
    TPC_CUDA(h, cudaMemcpy2DAsync(oh->trk_cov, 4 * (size_t)oh->cap_tracks, od.trk_cov, 4 * (size_t)od.cap_tracks, n4, 15,
                                  cudaMemcpyDeviceToHost, st));
  TPC_CUDA(h, back(oh->trk_cl_offset, od.trk_cl_offset, 4 * (size_t)(nt + 1)));
  if (status->status == TPC_OK) TPC_CUDA(h, back(oh->trk_cl_index, od.trk_cl_index, 4 * (size_t)nc));
  TPC_CUDA(h, cudaStreamSynchronize(st));
  return TPC_OK;
}

// ---- double-buffered host path: tpcSubmitHost / tpcCollectHost -------------------------------------------------
namespace {
// make slot `s` the active per-run state of the handle (0 = the synchronous path, 1 / 2 = the two pipeline slots)
int useSlot(tpcHandle* h, int s) {
  if (s == h->cur_slot) return TPC_OK;
  tpcHandle::Slot& o = h->slots[h->cur_slot];
  o.init = true;
  o.d_cnt = h->d_cnt; o.h_cnt = h->h_cnt; o.ev_done = h->ev_done; o.launches = h->launches; o.pending = h->pending;
  o.last_n = h->last_n;
  memcpy(o.pool, h->pool, sizeof(o.pool)); memcpy(o.pool_bytes, h->pool_bytes, sizeof(o.pool_bytes));
  tpcHandle::Slot& n = h->slots[s];
  if (!n.init) {
    TPC_CUDA(h, cudaMalloc(&n.d_cnt, 8 * (CNT_COUNT + 1)));
    TPC_CUDA(h, cudaMallocHost(&n.h_cnt, 8 * (CNT_COUNT + 1)));
    TPC_CUDA(h, cudaEventCreate(&n.ev_done));
    TPC_CUDA(h, cudaStreamCreateWithFlags(&n.stream, cudaStreamNonBlocking));
    TPC_CUDA(h, cudaEventCreate(&n.ev_begin));
    TPC_CUDA(h, cudaEventCreate(&n.ev_kernels));
    memset(n.h_cnt, 0, 8 * (CNT_COUNT + 1));
    n.init = true;
  }
  h->d_cnt = n.d_cnt; h->h_cnt = n.h_cnt; h->ev_done = n.ev_done; h->launches = n.launches; h->pending = n.pending;
  h->last_n = n.last_n;
  memcpy(h->pool, n.pool, sizeof(n.pool)); memcpy(h->pool_bytes, n.pool_bytes, sizeof(n.pool_bytes));
  h->cur_slot = s;
  return TPC_OK;
}
}  // namespace

extern "C" int tpcSubmitHost(tpcHandle* h, int slot, int64_t N, const uint32_t* row_offset, const float* y, const float* z,
                             const tpcTracks* oh) {
  if (!h || slot < 0 || slot > 1 || !row_offset || !oh || N < 0 || N >= (1ll << 31) || (N > 0 && (!y || !z)))
    return TPC_ERR_INVALID_ARG;
  if (oh->link_up_raw || oh->link_dn_raw || oh->link_up || oh->link_dn || oh->start_hits || oh->tl_status || oh->tl_nhits ||
      oh->tl_first_row || oh->tl_last_row || oh->tl_rowhit || oh->tl_x || oh->tl_par || oh->tl_cov || oh->tl_chi2 ||
      oh->trk_rf_status || oh->trk_mg_next || oh->trk_leg_partner || oh->trk_leg_chi2 || oh->cl_flags || oh->cl_owner || oh->cl_qcode || oh->cl_res_y || oh->cl_res_z || oh->cl_pos_code || oh->cl_res_code || oh->trk_mt_id || oh->trk_mt_rank || oh->mt_cl_offset || oh->mt_cl_index || !oh->trk_cl_offset || oh->cap_tracks < 0 || oh->cap_track_clusters < 0)
    return TPC_ERR_INVALID_ARG;
  TPC_CUDA(h, cudaSetDevice(h->device));
  int rc;
  if ((rc = useSlot(h, slot + 1))) return rc;
  tpcHandle::Slot& S = h->slots[slot + 1];
  if (S.submitted) { useSlot(h, 0); return TPC_ERR_INVALID_ARG; }      // collect first
  cudaStream_t st = S.stream;
  const int nb = h->P.n_buckets;
  const int64_t capT = std::max<int64_t>(std::max<int64_t>(4096, N / 8), h->hint_T);
  const int64_t capK = std::max<int64_t>(std::max<int64_t>(4096, N / 64), h->hint_K);
  const int64_t capC = std::max<int64_t>(std::max<int64_t>(N / 2, 1), h->hint_C);
  void *d_off, *d_y, *d_z, *ws;
  size_t wsb = 0;
  auto fail = [&](int code) { useSlot(h, 0); return code; };
  if ((rc = poolGet(h, 0, 4 * (size_t)(nb + 1), &d_off)) || (rc = poolGet(h, 1, 4 * (size_t)N, &d_y)) ||
      (rc = poolGet(h, 2, 4 * (size_t)N, &d_z)) || (rc = tpcWorkspaceBytes(h, N, capT, &wsb)) || (rc = poolGet(h, 3, wsb, &ws)))
    return fail(rc);
  void* p[11];
  const size_t K = (size_t)capK;
  const size_t sz[11] = {4 * K, 4 * K, 4 * K, 4 * K, 4 * K, 4 * K, 20 * K, 60 * K, 4 * K, 4 * (K + 1), 4 * (size_t)capC};
  for (int i = 0; i < 11; ++i)
    if ((rc = poolGet(h, 4 + i, sz[i], &p[i]))) return fail(rc);
  cudaEventRecord(S.ev_begin, st);
  if (cudaMemcpyAsync(d_off, row_offset, 4 * (size_t)(nb + 1), cudaMemcpyHostToDevice, st) != cudaSuccess ||
      (N > 0 && (cudaMemcpyAsync(d_y, y, 4 * (size_t)N, cudaMemcpyHostToDevice, st) != cudaSuccess ||
                 cudaMemcpyAsync(d_z, z, 4 * (size_t)N, cudaMemcpyHostToDevice, st) != cudaSuccess)))
    return fail(TPC_ERR_CUDA);
  // The kernels of this event start when those of the other slot's event are done (its copies out then overlap these
  // kernels, and the copies in above overlapped its kernels): without the order the two events would share the SMs
  // and finish together, copies and kernels never overlapping.
  {
    tpcHandle::Slot& O = h->slots[2 - slot];
    if (O.submitted && cudaStreamWaitEvent(st, O.ev_kernels, 0) != cudaSuccess) return fail(TPC_ERR_CUDA);
  }
  tpcTracks od{};
  od.cap_tracks = capK; od.cap_track_clusters = capC;
  od.trk_tracklet = (int32_t*)p[0]; od.trk_sector = (int32_t*)p[1]; od.trk_first_row = (int32_t*)p[2];
  od.trk_last_row = (int32_t*)p[3]; od.trk_ncl = (int32_t*)p[4]; od.trk_x = (float*)p[5]; od.trk_par = (float*)p[6];
  od.trk_cov = (float*)p[7]; od.trk_chi2 = (float*)p[8]; od.trk_cl_offset = (uint32_t*)p[9];
  od.trk_cl_index = (uint32_t*)p[10];
  const tpcClusters in{N, (const uint32_t*)d_off, nullptr, (const float*)d_y, (const float*)d_z, nullptr};
  if ((rc = tpcRun(h, &in, &od, capT, ws, h->pool_bytes[3], st))) return fail(rc);
  cudaEventRecord(S.ev_kernels, st);
  // The counts are not known on the host yet: copy back up to the capacities (the hints sit a few percent above the
  // last counts), tpcCollectHost trims.  tpcRun's own status copy and event come before these copies on the stream,
  // so a second event closes the slot.
  const int64_t nt = std::min<int64_t>(capK, oh->cap_tracks), nc = std::min<int64_t>(capC, oh->cap_track_clusters);
  const size_t n4 = 4 * (size_t)nt;
  auto back = [&](void* dst, const void* src, size_t bytes) {
    return (dst && bytes) ? cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st) : cudaSuccess;
  };
  bool ok = back(oh->trk_tracklet, od.trk_tracklet, n4) == cudaSuccess && back(oh->trk_sector, od.trk_sector, n4) == cudaSuccess &&
            back(oh->trk_first_row, od.trk_first_row, n4) == cudaSuccess && back(oh->trk_last_row, od.trk_last_row, n4) == cudaSuccess &&
            back(oh->trk_ncl, od.trk_ncl, n4) == cudaSuccess && back(oh->trk_x, od.trk_x, n4) == cudaSuccess &&
            back(oh->trk_chi2, od.trk_chi2, n4) == cudaSuccess;
  if (ok && nt > 0 && oh->trk_par)
    ok = cudaMemcpy2DAsync(oh->trk_par, 4 * (size_t)oh->cap_tracks, od.trk_par, 4 * (size_t)capK, n4, 5, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  if (ok && nt > 0 && oh->trk_cov)
    ok = cudaMemcpy2DAsync(oh->trk_cov, 4 * (size_t)oh->cap_tracks, od.trk_cov, 4 * (size_t)capK, n4, 15, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  ok = ok && back(oh->trk_cl_offset, od.trk_cl_offset, 4 * (size_t)(std::min<int64_t>(nt, oh->cap_tracks) + 1)) == cudaSuccess &&
       back(oh->trk_cl_index, od.trk_cl_index, 4 * (size_t)nc) == cudaSuccess &&
       cudaEventRecord(h->ev_done, st) == cudaSuccess;
  if (!ok) return fail(TPC_ERR_CUDA);
  S.submitted = true; S.capK = capK; S.capC = capC; S.oh = *oh;
  return useSlot(h, 0);
}

extern "C" int tpcCollectHost(tpcHandle* h, int slot, tpcRunStatus* status) {
  if (!h || slot < 0 || slot > 1 || !status) return TPC_ERR_INVALID_ARG;
  tpcHandle::Slot& S = h->slots[slot + 1];
  if (!S.submitted) return TPC_ERR_INVALID_ARG;
  TPC_CUDA(h, cudaSetDevice(h->device));
  int rc;
  if ((rc = useSlot(h, slot + 1))) return rc;
  rc = tpcGetRunStatus(h, status);            // waits for the slot's last event: run and copies are complete
  S.submitted = false;
  if (rc == TPC_OK) {
    // the per-stage events belong to the handle, not to the slot: with two events in flight they may be the other
    // slot's.  Per-stage times are valid for tpcRun / tpcRunHost only.
    memset(status->stage_ms, 0, sizeof(status->stage_ms));
    status->merge_ms = status->flags_ms = status->pack_ms = status->legs_ms = status->merged_ms = 0.0f;
    float ms = 0;
    if (cudaEventElapsedTime(&ms, S.ev_begin, S.ev_kernels) == cudaSuccess) status->submit_ms[0] = ms;
    if (cudaEventElapsedTime(&ms, S.ev_begin, h->ev_done) == cudaSuccess) status->submit_ms[1] = ms;
    if (status->status == TPC_OK &&
        (status->n_tracks > std::min(S.capK, S.oh.cap_tracks) || status->n_track_clusters > std::min(S.capC, S.oh.cap_track_clusters)))
      status->status = TPC_ERR_CAPACITY;
    // the next submission gets the capacities right (also after TPC_ERR_CAPACITY: the caller re-runs with tpcRunHost)
    h->hint_T = std::max(h->hint_T, status->n_start_hits + status->n_start_hits / 16);
    h->hint_K = std::max(h->hint_K, status->n_tracks + status->n_tracks / 16);
    h->hint_C = std::max(h->hint_C, status->n_track_clusters + status->n_track_clusters / 16);
  }
  const int rc2 = useSlot(h, 0);
  return rc ? rc : rc2;
}
