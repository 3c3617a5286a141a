// tpcca_start_hits_noalloc (include/tpcca.h): S4 start-hit selection for callers that must
// not allocate device memory.
//
// Who that is: a reconstruction step inside an online framework that claimed the GPU's memory once, as one
// slab, when the run started -- nothing is left for a cudaMalloc, and cudaMalloc / cudaFree stall every
// stream of the device while other time frames are in flight; a plug-in under a caching allocator (PyTorch's),
// which cannot see, reuse or account for memory taken behind its back; a QA hook that holds two link arrays
// and no tpcca context.  tpcca_create serves none of them: it wants a workspace sized by
// tpcca_workspace_bytes and itself creates events, a copy stream and pinned host memory.
//
// The stage needs scratch: one start-hit count and one output offset per 2048-cluster tile.  Here that scratch
// is a fixed array inside the library image (g_noalloc_scratch, 64 KiB).  Every GPU that loads libtpcca.so
// carries these 64 KiB from module load until the process exits; in exchange this entry point calls no
// cudaMalloc, cudaFree, cudaMallocHost, no stream / event creation and no library routine that allocates.
//
// Product code: no oracle code here; shares block_exclusive_scan with the other kernels (tpcca_dev.cuh).
// The existing path (k_clean_links + k_scan_pairs + k_start_hits in k_links.cuh) is untouched.
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "tpcca_dev.cuh"

namespace {

constexpr int kTile = 2048;                                            // clusters per tile = 256 threads x 8
constexpr int kMaxTiles = TPCCA_NOALLOC_MAX_CLUSTERS / kTile;          // 8192
constexpr int kMaxDevices = 64;
static_assert(TPCCA_NOALLOC_MAX_CLUSTERS % kTile == 0, "the limit is a whole number of tiles");
static_assert(kMaxTiles <= 1024 * 8, "k_na_scan covers at most 1024 threads x 8 tiles");

// The scratch.  [0, kMaxTiles): start hits per tile (written by k_na_count); [kMaxTiles, 2 kMaxTiles): first
// output slot of each tile (written by k_na_scan).  ONE array per device for the whole process: every call
// reuses it and finds the previous call's numbers in it.  Nothing in it has to start at zero -- each call
// overwrites entries [0, n_tiles) of both halves before it reads them and never reads beyond n_tiles -- so
// there is no clearing pass.  Two calls that are on the same GPU at the same time (different streams, or
// different host threads) would overwrite each other's counts: see the header.
//
// In HOST code the name g_noalloc_scratch is only a handle of the symbol, not a device address; the address a
// kernel can use comes from cudaGetSymbolAddress (scratch_of_device below), per device.
static __device__ __align__(256) int32_t g_noalloc_scratch[2 * kMaxTiles];

__device__ __forceinline__ bool is_start_hit(const int32_t* __restrict__ up, const int32_t* __restrict__ dn, int64_t p, int64_t n) {
  return p < n && dn[p] == -1 && up[p] >= 0;       // DESIGN.md 3.4 on the cleaned links
}

// tile_cnt[t] = number of start hits among positions [2048 t, 2048 t + 2048)
__global__ void __launch_bounds__(256)
k_na_count(const int32_t* __restrict__ up, const int32_t* __restrict__ dn, int64_t n, int32_t* __restrict__ tile_cnt) {
  const int64_t p0 = (int64_t)blockIdx.x * kTile;
  int cnt = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) cnt += __syncthreads_count(is_start_hit(up, dn, p0 + k * 256 + threadIdx.x, n));
  if (threadIdx.x == 0) tile_cnt[blockIdx.x] = cnt;
}

// tile_off[t] = sum of tile_cnt[0..t); *n_start = total.  One block; thread i owns tiles 8 i .. 8 i + 7.
__global__ void __launch_bounds__(1024)
k_na_scan(const int32_t* __restrict__ tile_cnt, int32_t* __restrict__ tile_off, int n_tiles, int32_t* __restrict__ n_start) {
  __shared__ int ws[33];
  int c[8], sum = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int t = threadIdx.x * 8 + k;
    c[k] = t < n_tiles ? tile_cnt[t] : 0;
    sum += c[k];
  }
  int total;
  int o = tpcca::block_exclusive_scan<int>(sum, ws, total);
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int t = threadIdx.x * 8 + k;
    if (t < n_tiles) tile_off[t] = o;
    o += c[k];
  }
  if (threadIdx.x == 0) *n_start = total;
}

// Ordered compaction.  Warp w of a tile owns the 256 consecutive positions [p0 + 256 w, p0 + 256 w + 256) in
// 8 coalesced rounds of 32; ballots give every start hit its rank, so slots ascend with the position.
__global__ void __launch_bounds__(256)
k_na_compact(const int32_t* __restrict__ up, const int32_t* __restrict__ dn, int64_t n,
             const int32_t* __restrict__ tile_off, int64_t cap, int32_t* __restrict__ start_hit) {
  __shared__ int warp_cnt[8];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t p0 = (int64_t)blockIdx.x * kTile + w * 256;
  unsigned m[8];
  int cnt = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    m[k] = __ballot_sync(0xffffffffu, is_start_hit(up, dn, p0 + k * 32 + lane, n));
    cnt += __popc(m[k]);
  }
  if (lane == 0) warp_cnt[w] = cnt;
  __syncthreads();
  int64_t o = tile_off[blockIdx.x];
  for (int i = 0; i < w; ++i) o += warp_cnt[i];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    if (m[k] & (1u << lane)) {
      const int64_t slot = o + __popc(m[k] & ((1u << lane) - 1u));
      if (slot < cap) start_hit[slot] = (int32_t)(p0 + k * 32 + lane);
    }
    o += __popc(m[k]);
  }
}

int fail(char* msg, size_t len, int code, const char* fmt, ...) {
  if (msg && len) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(msg, len, fmt, ap);
    va_end(ap);
  }
  return code;
}

// Device address of g_noalloc_scratch on `dev`, which must be the current device.  Resolved once per device
// (this is the set-up step: it makes the runtime load the library's module on that device if it has not yet).
std::mutex g_mu;
int32_t* g_scratch_addr[kMaxDevices];
cudaError_t scratch_of_device(int dev, int32_t** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    int32_t* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    g_scratch_addr[dev] = ptr;
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" int tpcca_start_hits_noalloc(int cuda_device, void* cuda_stream, const int32_t* link_up, const int32_t* link_dn,
                                        int64_t n_clusters, int32_t* start_hit, int64_t max_start_hits, int32_t* n_start,
                                        char* err_msg, size_t err_msg_len) {
  if (err_msg && err_msg_len) err_msg[0] = 0;
  // host-only checks first: a refused call touches neither the device nor the scratch
  if (n_clusters < 0 || max_start_hits < 0) return fail(err_msg, err_msg_len, TPCCA_E_ARG, "n_clusters and max_start_hits must be >= 0");
  if (n_clusters > (int64_t)TPCCA_NOALLOC_MAX_CLUSTERS)
    return fail(err_msg, err_msg_len, TPCCA_E_ARG,
                "n_clusters %lld exceeds TPCCA_NOALLOC_MAX_CLUSTERS %d (the fixed scratch of this entry point); split the call "
                "or use tpcca_run with a workspace", (long long)n_clusters, TPCCA_NOALLOC_MAX_CLUSTERS);
  if (!n_start) return fail(err_msg, err_msg_len, TPCCA_E_ARG, "n_start is NULL");
  if (n_clusters > 0 && (!link_up || !link_dn)) return fail(err_msg, err_msg_len, TPCCA_E_ARG, "link_up / link_dn is NULL");
  if (max_start_hits > 0 && !start_hit) return fail(err_msg, err_msg_len, TPCCA_E_ARG, "start_hit is NULL");
  if (cuda_device < 0 || cuda_device >= kMaxDevices) return fail(err_msg, err_msg_len, TPCCA_E_ARG, "cuda_device must be in 0..%d", kMaxDevices - 1);

  int prev = -1;
  cudaError_t e = cudaGetDevice(&prev);
  if (e != cudaSuccess) return fail(err_msg, err_msg_len, TPCCA_E_CUDA, "no usable CUDA device (%s); tpcca has no CPU path", cudaGetErrorString(e));
  if (prev != cuda_device && (e = cudaSetDevice(cuda_device)) != cudaSuccess)
    return fail(err_msg, err_msg_len, TPCCA_E_CUDA, "cudaSetDevice(%d) failed: %s", cuda_device, cudaGetErrorString(e));

  int rc = TPCCA_OK;
  int32_t* scratch = nullptr;
  if ((e = scratch_of_device(cuda_device, &scratch)) != cudaSuccess) {
    rc = fail(err_msg, err_msg_len, TPCCA_E_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch) on device %d failed: %s", cuda_device, cudaGetErrorString(e));
  } else {
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int n_tiles = (int)((n_clusters + kTile - 1) / kTile);
    int32_t* tile_cnt = scratch;
    int32_t* tile_off = scratch + kMaxTiles;
    if (n_tiles) k_na_count<<<n_tiles, 256, 0, st>>>(link_up, link_dn, n_clusters, tile_cnt);
    k_na_scan<<<1, 1024, 0, st>>>(tile_cnt, tile_off, n_tiles, n_start);      // n_tiles == 0: writes *n_start = 0
    if (n_tiles) k_na_compact<<<n_tiles, 256, 0, st>>>(link_up, link_dn, n_clusters, tile_off, max_start_hits, start_hit);
    if ((e = cudaGetLastError()) != cudaSuccess)
      rc = fail(err_msg, err_msg_len, TPCCA_E_CUDA, "tpcca_start_hits_noalloc: launch failed: %s", cudaGetErrorString(e));
  }
  if (prev != cuda_device) cudaSetDevice(prev);
  return rc;
}
