// tpc_noalloc.cu -- the one entry point of libtpcgpu.so that allocates nothing: tpcStartHitsNoAlloc (include/tpc_abi.h).
//
// What it computes: the a3 start-hit list (O3, R8; PAPER.md L83 track finding) from the
// cleaned links: cluster c is a start hit <=> link_dn[c] == -1 and link_up[c] != -1; the list is in ascending global
// input index.  It is the stream compaction of tpc_links.cuh (startCount -> scan of the tile counts -> startWrite) reading
// the links in their exported form (global input indices, as tpcTracks.link_up / link_dn) instead of the library's
// internal spos_by_orig array.  The scratch of that compaction -- one count per tile of NA_TILE clusters -- lives in the
// file-scope device array g_scratch below instead of the caller's workspace, so callers that cannot call cudaMalloc
// (code under CUDA graph capture, tight serving loops) need no workspace at all.
//
// Rules this file keeps
//   - g_scratch is a `static __device__` array: every GPU that loads the library holds its NA_SCRATCH_BYTES (33 KB) until
//     exit.  In HOST code the name g_scratch is a host-side stand-in, not a device address; the address the kernels get
//     comes from cudaGetSymbolAddress, once per device with that device current (scratchOf), and is checked.
//   - no cudaMalloc / cudaFree / allocating library routine anywhere in this file; sizes beyond TPC_NOALLOC_MAX_CLUSTERS
//     are refused with TPC_ERR_NOALLOC_LIMIT before anything is launched.
//   - every call shares the array and finds the last call's contents in it.  Nothing has to start at zero: phase 1
//     writes the counts of tiles [0, ntiles), phase 2 reads exactly those and writes the header word, phase 3 reads
//     exactly those; words beyond ntiles left by a larger earlier call are never read.  (The header is still cleared
//     by phase 2 of every call, n == 0 included, so that a stale total can never be taken for this call's.)
//   - calls that overlap on the GPU (two streams, two host threads, two graphs in flight) race on the array.  Calls
//     enqueued on one stream, or otherwise ordered on the device, are safe.
// This translation unit shares no code with tpc_api.cu and changes none of its paths.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/tpc_abi.h"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_ITEMS = 8;
constexpr int NA_TILE = NA_THREADS * NA_ITEMS;                                     // 2048 clusters per tile
constexpr int64_t NA_MAX_CLUSTERS = TPC_NOALLOC_MAX_CLUSTERS;                       // 2^24
constexpr int NA_MAX_TILES = (int)((NA_MAX_CLUSTERS + NA_TILE - 1) / NA_TILE);      // 8192
constexpr int NA_HEADER_WORDS = 64;                                                 // 256 bytes: [0..1] = total of the last call
constexpr int NA_SCRATCH_WORDS = NA_HEADER_WORDS + NA_MAX_TILES;
constexpr size_t NA_SCRATCH_BYTES = 4 * (size_t)NA_SCRATCH_WORDS;                   // 33 024 bytes
constexpr int NA_MAX_DEVICES = 64;

static __device__ __align__(256) uint32_t g_scratch[NA_SCRATCH_WORDS];
static_assert(sizeof(g_scratch) == NA_SCRATCH_BYTES && NA_SCRATCH_BYTES == 33024, "the size include/tpc_abi.h states");

// exclusive scan of one value per thread over the block (blockDim.x a multiple of 32, at most 1024); *total = block sum
__device__ __forceinline__ uint32_t blockScan(uint32_t v, uint32_t* sm, uint32_t* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t o = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane >= d) inc += o;
  }
  if (lane == 31) sm[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    const uint32_t w = lane < nwarp ? sm[lane] : 0u;
    uint32_t winc = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t o = __shfl_up_sync(0xffffffffu, winc, d);
      if (lane >= d) winc += o;
    }
    sm[lane] = winc - w;
    if (lane == 31) sm[32] = winc;
  }
  __syncthreads();
  const uint32_t ex = sm[warp] + inc - v;
  *total = sm[32];
  __syncthreads();
  return ex;
}

// the NA_ITEMS consecutive clusters of one thread: bit k of the result = cluster first + k is a start hit
__device__ __forceinline__ uint32_t startMask(int64_t N, const int32_t* __restrict__ up, const int32_t* __restrict__ dn,
                                              int64_t first, bool aligned) {
  uint32_t m = 0;
  if (aligned && first + NA_ITEMS <= N) {
    int32_t u[NA_ITEMS], d[NA_ITEMS];
#pragma unroll
    for (int k = 0; k < NA_ITEMS; k += 4) {
      const int4 qu = *reinterpret_cast<const int4*>(up + first + k);
      const int4 qd = *reinterpret_cast<const int4*>(dn + first + k);
      u[k] = qu.x; u[k + 1] = qu.y; u[k + 2] = qu.z; u[k + 3] = qu.w;
      d[k] = qd.x; d[k + 1] = qd.y; d[k + 2] = qd.z; d[k + 3] = qd.w;
    }
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k)
      if (d[k] == -1 && u[k] != -1) m |= 1u << k;
  } else {
#pragma unroll
    for (int k = 0; k < NA_ITEMS; ++k)
      if (first + k < N && dn[first + k] == -1 && up[first + k] != -1) m |= 1u << k;
  }
  return m;
}

// phase 1: start hits per tile -> scratch
__global__ void __launch_bounds__(NA_THREADS) noallocStartCount(int64_t N, const int32_t* __restrict__ up,
                                                                const int32_t* __restrict__ dn, int aligned,
                                                                uint32_t* __restrict__ tile_cnt) {
  __shared__ uint32_t sm[33];
  const int64_t first = (int64_t)blockIdx.x * NA_TILE + (int64_t)threadIdx.x * NA_ITEMS;
  const uint32_t c = __popc(startMask(N, up, dn, first, aligned != 0));
  uint32_t total;
  blockScan(c, sm, &total);
  if (threadIdx.x == 0) tile_cnt[blockIdx.x] = total;
}

// phase 2, one block: tile counts -> exclusive tile offsets in place; the total goes to the header and to *n_out.
// Runs for ntiles == 0 as well: it is what clears the header of the last call.
__global__ void __launch_bounds__(1024) noallocTileScan(uint32_t* __restrict__ header, uint32_t* __restrict__ tile_cnt,
                                                        int ntiles, int64_t* __restrict__ n_out) {
  __shared__ uint32_t sm[33];
  if (threadIdx.x < 2) header[threadIdx.x] = 0;
  uint32_t carry = 0;
  for (int base = 0; base < ntiles; base += blockDim.x) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < ntiles ? tile_cnt[i] : 0u;
    uint32_t total;
    const uint32_t ex = blockScan(v, sm, &total);
    if (i < ntiles) tile_cnt[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0) {
    header[0] = carry;
    *n_out = (int64_t)carry;
  }
}

// phase 3: the global indices of the start hits, ascending, truncated at cap
__global__ void __launch_bounds__(NA_THREADS) noallocStartWrite(int64_t N, const int32_t* __restrict__ up,
                                                                const int32_t* __restrict__ dn, int aligned,
                                                                const uint32_t* __restrict__ tile_off, int64_t cap,
                                                                uint32_t* __restrict__ start_hits) {
  __shared__ uint32_t sm[33];
  const int64_t first = (int64_t)blockIdx.x * NA_TILE + (int64_t)threadIdx.x * NA_ITEMS;
  const uint32_t m = startMask(N, up, dn, first, aligned != 0);
  uint32_t total;
  uint32_t o = blockScan(__popc(m), sm, &total) + tile_off[blockIdx.x];
#pragma unroll
  for (int k = 0; k < NA_ITEMS; ++k)
    if (m >> k & 1u) {
      if ((int64_t)o < cap) start_hits[o] = (uint32_t)(first + k);
      ++o;
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------------
std::mutex g_mu;
uint32_t* g_scratch_dev[NA_MAX_DEVICES] = {};      // device address of g_scratch per CUDA device, NULL = not set up yet
thread_local char g_msg[256] = "";

int fail(int code, const char* what, cudaError_t e) {
  snprintf(g_msg, sizeof g_msg, "%s: %s", what, cudaGetErrorString(e));
  return code;
}

struct DeviceScope {          // makes `dev` current for the scope and puts the caller's device back
  int prev = -1;
  cudaError_t err;
  explicit DeviceScope(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
  }
  ~DeviceScope() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

// The device address of g_scratch on `dev` (current).  Looked up once per device; never the host-side symbol itself.
int scratchOf(int dev, uint32_t** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_dev[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_scratch);
    if (e != cudaSuccess) return fail(TPC_ERR_CUDA, "cudaGetSymbolAddress(g_scratch)", e);
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255) != 0) {
      snprintf(g_msg, sizeof g_msg, "cudaGetSymbolAddress(g_scratch) returned %p: not a 256-byte aligned device address", p);
      return TPC_ERR_CUDA;
    }
    cudaPointerAttributes a;
    const cudaError_t ea = cudaPointerGetAttributes(&a, p);
    if (ea != cudaSuccess) return fail(TPC_ERR_CUDA, "cudaPointerGetAttributes(scratch)", ea);
    if (a.type != cudaMemoryTypeDevice || a.device != dev) {
      snprintf(g_msg, sizeof g_msg, "scratch address %p is not device memory of device %d (type %d, device %d)", p, dev,
               (int)a.type, a.device);
      return TPC_ERR_CUDA;
    }
    g_scratch_dev[dev] = static_cast<uint32_t*>(p);
  }
  *out = g_scratch_dev[dev];
  return TPC_OK;
}

}  // namespace

extern "C" {

int64_t tpcNoAllocMaxClusters(void) { return NA_MAX_CLUSTERS; }

const char* tpcNoAllocLastError(void) { return g_msg; }

int tpcNoAllocSetup(int cuda_device) {
  g_msg[0] = 0;
  if (cuda_device < 0 || cuda_device >= NA_MAX_DEVICES) {
    snprintf(g_msg, sizeof g_msg, "cuda_device %d outside [0, %d)", cuda_device, NA_MAX_DEVICES);
    return TPC_ERR_INVALID_ARG;
  }
  DeviceScope scope(cuda_device);
  if (scope.err != cudaSuccess) return fail(TPC_ERR_CUDA, "cudaSetDevice", scope.err);
  uint32_t* s = nullptr;
  return scratchOf(cuda_device, &s);
}

int tpcStartHitsNoAlloc(int cuda_device, int64_t n_clusters, const int32_t* link_up, const int32_t* link_dn,
                        uint32_t* start_hits, int64_t cap_start_hits, int64_t* n_start_hits, void* cuda_stream) {
  g_msg[0] = 0;
  if (cuda_device < 0 || cuda_device >= NA_MAX_DEVICES || n_clusters < 0 || cap_start_hits < 0 || !n_start_hits ||
      (n_clusters > 0 && (!link_up || !link_dn)) || (cap_start_hits > 0 && !start_hits)) {
    snprintf(g_msg, sizeof g_msg, "NULL pointer, negative size or cuda_device outside [0, %d)", NA_MAX_DEVICES);
    return TPC_ERR_INVALID_ARG;
  }
  if (n_clusters > NA_MAX_CLUSTERS) {
    snprintf(g_msg, sizeof g_msg, "n_clusters %lld exceeds TPC_NOALLOC_MAX_CLUSTERS %lld: the static scratch holds %d tile counts",
             (long long)n_clusters, (long long)NA_MAX_CLUSTERS, NA_MAX_TILES);
    return TPC_ERR_NOALLOC_LIMIT;
  }
  DeviceScope scope(cuda_device);
  if (scope.err != cudaSuccess) return fail(TPC_ERR_CUDA, "cudaSetDevice", scope.err);
  uint32_t* scratch = nullptr;
  const int rc = scratchOf(cuda_device, &scratch);
  if (rc != TPC_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  uint32_t* tile = scratch + NA_HEADER_WORDS;
  const int ntiles = (int)((n_clusters + NA_TILE - 1) / NA_TILE);
  const int aligned = ((reinterpret_cast<uintptr_t>(link_up) | reinterpret_cast<uintptr_t>(link_dn)) & 15) == 0;
  if (ntiles > 0) noallocStartCount<<<ntiles, NA_THREADS, 0, st>>>(n_clusters, link_up, link_dn, aligned, tile);
  noallocTileScan<<<1, 1024, 0, st>>>(scratch, tile, ntiles, n_start_hits);
  if (ntiles > 0 && cap_start_hits > 0)
    noallocStartWrite<<<ntiles, NA_THREADS, 0, st>>>(n_clusters, link_up, link_dn, aligned, tile, cap_start_hits, start_hits);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(TPC_ERR_CUDA, "kernel launch", e);
  return TPC_OK;
}

}  // extern "C"
