// Host side of the tpcca C-ABI (include/tpcca.h): workspace carving, stage scheduling on the
// caller's stream, per-stage CUDA events, error mapping.  No torch types, no CPU compute path:
// every stage of the hot path runs in the kernels of k_grid.cuh / k_links.cuh / k_tracklets.cuh.
#include <chrono>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <algorithm>
#include <utility>
#include <vector>

#include "k_merge.cuh"

using namespace tpcca;

namespace {

thread_local std::string g_last_error;

constexpr size_t kAlign = 256;
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

// ---- workspace layout -------------------------------------------------------------
struct Layout {
  size_t tables, sec, status, tot;
  size_t in_y, in_z, in_row;
  size_t syz, order, bin_start, row_start, nf_tile_start, nf_desc, cb_cnt, cb_start, big_list, rec, zorder, sh_first, sh_cnt, sh_blk, sh_pre, perm;
  size_t up_raw, dn_raw, up, dn;
  size_t tile_cnt, tile_off, start_bits;
  size_t start_hit, hits, trk_v, trk_n, hs;
  size_t o_x_ref, o_z_ref, o_chi2, o_par, o_cov, o_n_hits, o_n_fit, o_first, o_last, o_start, o_hit_offset, o_hit_idx;
  size_t sel_n_own, sel_track, slot_trk;   // S6 (its other buffers alias S1 / S5 scratch: see sel_out)
  size_t res;   // S7: tpcca_residual[N]
  size_t mg_out, mg_ok, mg_cnt, mg_cur, mg_list, mg_keys, mg_links;   // S8 (chain outputs alias the parked-tracklet buffer)
  int64_t mg_nzb;
  size_t total;
  int64_t n_tiles_max, nf_tiles_max, n_cb;
};

// S8 candidate index: z buckets of width max(mg_zpre, 8 cm, range / 4096) over the z range of the grid
int64_t mg_z_buckets(const tpcca_params* p, float* lo, float* inv) {
  double zmax = p->grid_z_lo;
  for (int r = 0; r < p->n_rows; ++r) zmax = std::max(zmax, (double)p->grid_z_lo + (double)p->grid_nz[r] / (double)p->grid_inv_bin_z[r]);
  const double range = std::max(zmax - (double)p->grid_z_lo, 1.0);
  const double width = std::max({(double)p->mg_zpre, 8.0, range / 4096.0});
  if (lo) *lo = p->grid_z_lo;
  if (inv) *inv = (float)(1.0 / width);
  return (int64_t)std::ceil(range / width) + 1;
}

int64_t bins_per_sector(const tpcca_params* p) {
  int64_t nb = 0;
  for (int r = 0; r < p->n_rows; ++r) nb += (int64_t)p->grid_ny[r] * p->grid_nz[r];
  return nb;
}

// S1 level 1: z slices per coarse bucket (log2).  Larger buckets amortise the per-block work of the level-2
// sort, but a bucket must fit its shared-memory buffers (kSortCapR clusters, kSortCapB bins): the largest shift
// that keeps the mean bucket at the context's capacity below ~700 clusters and every bucket within kSortCapB bins.
int slab_shift_for(const tpcca_params* p, int64_t N) {
  int ny_max = 1;
  for (int r = 0; r < p->n_rows; ++r) ny_max = std::max(ny_max, (int)p->grid_ny[r]);
  for (int sh = kSlabShiftMax; sh > kSlabShiftMin; --sh) {
    int64_t ncb = 0;
    for (int r = 0; r < p->n_rows; ++r) ncb += (p->grid_nz[r] + (1 << sh) - 1) >> sh;
    const double mean = (double)N / ((double)p->n_sectors * (double)std::max<int64_t>(ncb, 1));
    if (mean <= 700.0 && (int64_t)ny_max << sh <= kSortCapB) return sh;
  }
  return kSlabShiftMin;
}

Layout make_layout(const tpcca_params* p, int64_t N, int64_t CS) {
  Layout L{};
  const int kSlab = 1 << slab_shift_for(p, N);
  size_t cur = 0;
  auto take = [&](size_t bytes) { size_t o = cur; cur = align_up(cur + bytes); return o; };
  const int64_t ns = p->n_sectors, nr = p->n_rows, nb = bins_per_sector(p);
  L.n_tiles_max = std::max<int64_t>(N / 2048 + ns + 1, CS / 1024 + 2);
  L.n_cb = 0;
  for (int r = 0; r < p->n_rows; ++r) L.n_cb += (p->grid_nz[r] + kSlab - 1) / kSlab;
  L.tables = take(sizeof(DevTables));
  L.sec = take(sizeof(SectorDesc) * (kMaxSectors + 1));
  L.status = take(sizeof(DevStatus));
  L.tot = take(sizeof(int64_t) * 8);
  const size_t n_in = (size_t)N + 8 * kMaxSectors;   // every sector's copy starts 8-element aligned
  L.in_y = take(4 * n_in);
  L.in_z = take(4 * n_in);
  L.in_row = take(2 * n_in);
  L.syz = take(8 * (size_t)N + 64);                       // + pad: S2 stages 16-byte aligned runs
  L.order = take(4 * (size_t)N);
  L.bin_start = take(4 * (size_t)(ns * (nb + 1)) + 64);   // + pad (same reason)
  L.row_start = take(4 * (size_t)(ns * (nr + 1)));
  L.nf_tiles_max = N / kNfTile + ns * nr + 1;
  L.nf_tile_start = take(4 * (size_t)(ns * nr + 1));
  L.nf_desc = take(sizeof(NfTileDesc) * (size_t)L.nf_tiles_max);
  L.cb_cnt = take(4 * (size_t)(ns * (L.n_cb + 1)));
  L.cb_start = take(4 * (size_t)(ns * (L.n_cb + 1)));
  L.big_list = take(4 * (size_t)(ns * L.n_cb));
  L.rec = take(16 * (size_t)N);
  L.zorder = take(4 * (size_t)(2 * L.n_cb));   // [n_cb] buckets by ascending z, then [n_cb] bucket -> row | slab << 8
  L.sh_first = take(4 * (size_t)(ns * L.n_cb));
  L.sh_cnt = take(4 * (size_t)(ns * L.n_cb));
  L.sh_blk = take(sizeof(int2) * (size_t)(ns * L.n_cb / 256 + 2));
  L.sh_pre = take(sizeof(longlong2) * (size_t)(ns * L.n_cb / 256 + 2));
  L.perm = take(16 * (size_t)CS);      // int4 work records of S5
  L.up_raw = take(4 * (size_t)N);
  L.dn_raw = take(4 * (size_t)N);
  L.up = take(4 * (size_t)N);
  L.dn = take(4 * (size_t)N);
  L.tile_cnt = take(sizeof(int2) * (size_t)L.n_tiles_max);
  L.tile_off = take(sizeof(longlong2) * (size_t)L.n_tiles_max);
  L.start_bits = take(4 * 64 * (size_t)(N / 2048 + ns + 1));   // S3 -> S4: start-hit bitmap, 64 words per 2048-cluster tile
  L.start_hit = take(4 * (size_t)CS);
  L.hits = take(4 * (size_t)(nr * CS));
  L.trk_v = take(16 * (size_t)(kTrkV * CS));   // finished tracks: records of kTrkV 16-byte vectors
  L.trk_n = take(4 * (size_t)CS);             // n_hits per slot (0 = rejected)
  L.hs = take(16 * (size_t)(kHsV * CS) + 4 * (size_t)(ns + 1));   // parked tracklets: records of kHsV 16-byte vectors (S6: sel hit_offset)
  L.o_x_ref = take(4 * (size_t)CS);
  L.o_z_ref = take(4 * (size_t)CS);
  L.o_chi2 = take(4 * (size_t)CS);
  L.o_par = take(4 * (size_t)(5 * CS));
  L.o_cov = take(4 * (size_t)(15 * CS));
  L.o_n_hits = take(4 * (size_t)CS);
  L.o_n_fit = take(4 * (size_t)CS);
  L.o_first = take(4 * (size_t)CS);
  L.o_last = take(4 * (size_t)CS);
  L.o_start = take(4 * (size_t)CS);
  L.o_hit_offset = take(4 * (size_t)(CS + ns + 1));
  L.o_hit_idx = take(4 * (size_t)(nr * CS));
  L.sel_n_own = take(4 * (size_t)CS);
  L.sel_track = take(4 * (size_t)CS);
  L.slot_trk = take(4 * (size_t)CS);     // start-hit slot -> global track (S5 gather), -1 = rejected
  L.res = take(sizeof(tpcca_residual) * (size_t)N);
  L.mg_nzb = mg_z_buckets(p, nullptr, nullptr);
  L.mg_out = take(4 * (size_t)(6 * CS)); L.mg_ok = take(4 * (size_t)CS);
  L.mg_cnt = take(4 * (size_t)(ns * nr * L.mg_nzb + 2)); L.mg_cur = take(4 * (size_t)(ns * nr * L.mg_nzb + 2));
  L.mg_list = take(4 * (size_t)CS); L.mg_keys = take(8 * (size_t)(2 * CS)); L.mg_links = take(4 * (size_t)(4 * CS));
  L.total = cur;
  return L;
}

int check_params(const tpcca_params* p, std::string& err) {
  auto fail = [&](const char* m) { err = m; return TPCCA_E_ARG; };
  if (!p) return fail("params is NULL");
  if (p->n_sectors < 1 || p->n_sectors > TPCCA_MAX_SECTORS) return fail("n_sectors out of range");
  if (p->n_rows < 3 || p->n_rows > TPCCA_MAX_ROWS) return fail("n_rows out of range (3..TPCCA_MAX_ROWS)");
  if (!p->row_x || !p->grid_y_lo || !p->grid_inv_bin_y || !p->grid_ny || !p->grid_inv_bin_z || !p->grid_nz ||
      !p->nf_hy_up || !p->nf_hz_up || !p->nf_hy_dn || !p->nf_hz_dn || !p->nf_cut)
    return fail("a table pointer is NULL");
  int64_t nb = 0;
  for (int r = 0; r < p->n_rows; ++r) {
    if (p->grid_ny[r] < 1 || p->grid_nz[r] < 1) return fail("grid_ny / grid_nz must be >= 1");
    if (p->grid_ny[r] >= (1 << 24) || p->grid_nz[r] >= (1 << 24)) return fail("grid_ny / grid_nz must be < 2^24");
    if (r > 0 && !(p->row_x[r] > p->row_x[r - 1])) return fail("row_x must be strictly increasing");
    nb += (int64_t)p->grid_ny[r] * p->grid_nz[r];
  }
  if ((nb + 1) * (int64_t)p->n_sectors >= (int64_t)0xFFFFFFF0u) return fail("too many grid bins (n_sectors * (bins + 1) must fit 32 bits)");
  if (nb >= 0x7FFFFFF0) return fail("too many grid bins per sector");
  if (p->sel_max_shared_permille < 0 || p->sel_max_shared_permille > 1000) return fail("sel_max_shared_permille must be in 0..1000");
  if (!(p->res_inv_quantum > 0.0f)) return fail("res_inv_quantum must be > 0");
  if (p->sectors_per_side < 0 || p->mg_max_row_gap < 0) return fail("sectors_per_side / mg_max_row_gap must be >= 0");
  if (!(p->mg_dy > 0.0f) || !(p->mg_dz > 0.0f) || !(p->mg_dsin > 0.0f) || !(p->mg_zpre > 0.0f)) return fail("mg_dy / mg_dz / mg_dsin / mg_zpre must be > 0");
  return TPCCA_OK;
}

int64_t default_cap(int64_t N, int64_t CS) {
  if (CS <= 0) CS = N / 8 + 1024;
  if (CS > N / 2 + 1) CS = N / 2 + 1;
  if (CS < 1) CS = 1;
  return CS;
}

}  // namespace

struct tpcca_ctx {
  int device = 0;
  int sm_count = 148;
  int nf_blocks_per_sm = 3;
  bool nf_dense = false;               // S2 kernel instance with the deeper hit cache (tpcca_create)
  NfTable nftab{};                    // S2 per-row constants, passed to k_neighbours by value (constant bank)
  cudaStream_t stream = nullptr;
  cudaStream_t copy_stream = nullptr;  // D2H copies of tpcca_get_tracks(HOST): they wait only for the stage that made the data
  char* ws = nullptr;
  size_t ws_bytes = 0;
  int64_t N = 0, CS = 0;
  int ns = 0, nr = 0;
  int64_t nb = 0;
  Layout L{};
  DevTables tab{};
  // sectors
  struct Sec { bool loaded = false; int64_t n = 0; const float* y = nullptr; const float* z = nullptr; const uint16_t* row = nullptr; };
  std::vector<Sec> sec;
  int64_t in_used = 0;
  std::vector<SectorDesc> desc;       // as uploaded by the last run
  int64_t n_total = 0;
  int n_tiles256 = 0, n_tiles2048 = 0, max_tiles256 = 0;
  uint32_t done_mask = 0;             // stages whose outputs are valid for the loaded clusters
  bool desc_valid = false;
  static constexpr int kRing = 16;
  cudaEvent_t ev[kRing][9]{};
  MgParams mgp{};
  uint32_t ev_mask[kRing]{};          // stage mask of the run that used the slot (0 = unused)
  int64_t run_count = 0;
  char* arena = nullptr;              // pinned host arena of tpcca_get_tracks(HOST)
  size_t arena_bytes = 0;
  int64_t launches = 0;
  DevStatus status{};
  bool status_valid = false;
  std::string err;

  template <class Tp> Tp* at(size_t off) const { return reinterpret_cast<Tp*>(ws + off); }
};

namespace {

int set_err(tpcca_ctx* c, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (c) c->err = buf; else g_last_error = buf;
  return code;
}

#define CU(c, call)                                                                             \
  do {                                                                                          \
    cudaError_t e_ = (call);                                                                    \
    if (e_ != cudaSuccess) return set_err((c), TPCCA_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

// Every entry point that issues CUDA calls runs on the context's device and leaves the caller's current device
// as it found it (a host thread that serves several GPUs must not have its device switched under it).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  cudaError_t err = cudaSuccess;
  explicit DeviceGuard(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) { err = cudaSetDevice(dev); switched = (err == cudaSuccess); }
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
#define GUARD(c)                                                                                        \
  DeviceGuard guard_((c)->device);                                                                      \
  if (guard_.err != cudaSuccess) return set_err((c), TPCCA_E_CUDA, "cudaSetDevice(%d) failed: %s", (c)->device, cudaGetErrorString(guard_.err))

int fetch_status(tpcca_ctx* c);

int status_errors(tpcca_ctx* c) {
  if (c->status.err_range) return set_err(c, TPCCA_E_RANGE, "a cluster has row >= n_rows (%d)", c->nr);
  if (c->status.err_capacity)
    return set_err(c, TPCCA_E_WORKSPACE, "start-hit capacity exceeded: %d start hits > max_start_hits %lld",
                   c->status.n_start, (long long)c->CS);
  if (c->status.err_select) return set_err(c, TPCCA_E_WORKSPACE, "S6: a sector holds 2^23 or more tracks (selector key capacity)");
  return TPCCA_OK;
}

// Device status as of the end of stage `stage` (1..5) of the last run, without waiting for later stages:
// the copy stream waits for that stage's event only.  The start-hit fields are final after S4, the track
// fields after S5.
int fetch_status_after(tpcca_ctx* c, int stage) {
  if (c->run_count == 0) return fetch_status(c);
  const int k = (int)((c->run_count - 1) % tpcca_ctx::kRing);
  // The wait is taken on the HOST: a copy-stream entry that waits for the event would sit in a copy-engine queue
  // until the stage is done and hold up every copy another context has queued behind it on the same engine.
  CU(c, cudaEventSynchronize(c->ev[k][stage]));
  CU(c, cudaMemcpyAsync(&c->status, c->at<DevStatus>(c->L.status), sizeof(DevStatus), cudaMemcpyDeviceToHost, c->copy_stream));
  CU(c, cudaStreamSynchronize(c->copy_stream));
  return status_errors(c);
}

int fetch_status(tpcca_ctx* c) {
  // (never the legacy default stream: a synchronous cudaMemcpy would wait for every other context's work)
  CU(c, cudaMemcpyAsync(&c->status, c->at<DevStatus>(c->L.status), sizeof(DevStatus), cudaMemcpyDeviceToHost, c->stream));
  CU(c, cudaStreamSynchronize(c->stream));
  c->status_valid = true;
  return status_errors(c);
}

// S6 compact table of the selected tracks: 28 planes of CS words in the S5 slot-record buffer (trk_v: exactly
// 28 * 4 * CS bytes), its hit_offset in the parked-tracklet buffer (hs), its hit CSR in the per-tracklet hit lines
SelOut sel_out(const tpcca_ctx* c) {
  static_assert(kTrkV * 16 == 28 * 4, "the selected table's 28 planes fill the slot-record buffer exactly");
  const Layout& L = c->L;
  const size_t cs = (size_t)c->CS;
  float* f = c->at<float>(L.trk_v);
  int32_t* i32 = reinterpret_cast<int32_t*>(f);
  SelOut so;
  so.sel_track = c->at<int32_t>(L.sel_track);
  so.o.x_ref = f; so.o.z_ref = f + cs; so.o.chi2 = f + 2 * cs; so.o.par = f + 3 * cs; so.o.cov = f + 8 * cs;
  so.o.n_hits = i32 + 23 * cs; so.o.n_fit = i32 + 24 * cs; so.o.first_row = i32 + 25 * cs; so.o.last_row = i32 + 26 * cs;
  so.o.start_hit = i32 + 27 * cs;
  so.o.hit_offset = c->at<int32_t>(L.hs);
  so.o.hit_idx = c->at<int32_t>(L.hits);
  return so;
}

// S8 buffers; the per-chain outputs (29 planes of CS words) alias the parked-tracklet buffer behind the selected
// table's hit_offset (free after S5, like the rest of the S6 tables)
MgBuf mg_buf(const tpcca_ctx* c) {
  static_assert(kHsV * 16 >= 4 + 29 * 4 + 8, "chain outputs fit the parked-tracklet buffer");
  const Layout& L = c->L;
  const size_t cs = (size_t)c->CS;
  MgBuf b;
  b.out_x = c->at<float>(L.mg_out); b.out_p = b.out_x + cs; b.out_ok = c->at<int32_t>(L.mg_ok);
  b.bk_cnt = c->at<uint32_t>(L.mg_cnt); b.bk_list = c->at<int32_t>(L.mg_list);
  b.next_key = c->at<unsigned long long>(L.mg_keys); b.prev_key = b.next_key + cs;
  int32_t* l = c->at<int32_t>(L.mg_links);
  b.next_sec = l; b.next_trk = l + cs; b.prev_sec = l + 2 * cs; b.prev_trk = l + 3 * cs;
  char* base = c->ws + L.hs + align_up(4 * (cs + (size_t)c->ns + 1));
  int32_t* i32 = reinterpret_cast<int32_t*>(base);
  float* f = reinterpret_cast<float*>(base);
  b.n_seg = i32; b.n_hits = i32 + cs; b.n_fit = i32 + 2 * cs; b.first_row = i32 + 3 * cs; b.last_row = i32 + 4 * cs; b.frame_seg = i32 + 5 * cs;
  b.x_ref = f + 6 * cs; b.z_ref = f + 7 * cs; b.chi2 = f + 8 * cs; b.par = f + 9 * cs; b.cov = f + 14 * cs;
  return b;
}

}  // namespace

extern "C" {

const char* tpcca_version(void) { return "tpcca 0.2 (sm_100a)"; }

const char* tpcca_last_error(const tpcca_ctx* ctx) { return ctx ? ctx->err.c_str() : g_last_error.c_str(); }

int tpcca_workspace_bytes(const tpcca_params* params, int64_t max_clusters_total, int64_t max_start_hits,
                          size_t* out_bytes) {
  std::string e;
  int rc = check_params(params, e);
  if (rc) return set_err(nullptr, rc, "%s", e.c_str());
  if (!out_bytes || max_clusters_total < 0 || max_clusters_total >= 0x7FFFFF00)
    return set_err(nullptr, TPCCA_E_ARG, "max_clusters_total must be in [0, 2^31)");
  const int64_t N = std::max<int64_t>(max_clusters_total, 1);
  *out_bytes = make_layout(params, N, default_cap(N, max_start_hits)).total;
  return TPCCA_OK;
}

int tpcca_create(const tpcca_params* p, int cuda_device, void* cuda_stream, void* workspace, size_t workspace_bytes,
                 int64_t max_clusters_total, int64_t max_start_hits, tpcca_ctx** out_ctx) {
  if (!out_ctx) return set_err(nullptr, TPCCA_E_ARG, "out_ctx is NULL");
  *out_ctx = nullptr;
  std::string e;
  int rc = check_params(p, e);
  if (rc) return set_err(nullptr, rc, "%s", e.c_str());
  if (max_clusters_total < 0 || max_clusters_total >= 0x7FFFFF00)
    return set_err(nullptr, TPCCA_E_ARG, "max_clusters_total must be in [0, 2^31)");
  int n_dev = 0;
  cudaError_t ce = cudaGetDeviceCount(&n_dev);
  if (ce != cudaSuccess || n_dev <= 0)
    return set_err(nullptr, TPCCA_E_CUDA, "no usable CUDA device (%s); tpcca has no CPU path",
                   ce != cudaSuccess ? cudaGetErrorString(ce) : "device count 0");
  if (cuda_device < 0 || cuda_device >= n_dev) return set_err(nullptr, TPCCA_E_ARG, "cuda_device out of range");
  DeviceGuard guard(cuda_device);
  if (guard.err != cudaSuccess) return set_err(nullptr, TPCCA_E_CUDA, "cudaSetDevice(%d) failed: %s", cuda_device, cudaGetErrorString(guard.err));
  cudaDeviceProp prop;
  CU(nullptr, cudaGetDeviceProperties(&prop, cuda_device));
  if (prop.major != 10)
    return set_err(nullptr, TPCCA_E_CUDA, "device %d is sm_%d%d; this library holds sm_100a code only", cuda_device,
                   prop.major, prop.minor);
  const int64_t N = std::max<int64_t>(max_clusters_total, 1);
  const int64_t CS = default_cap(N, max_start_hits);
  Layout L = make_layout(p, N, CS);
  if (!workspace || ((uintptr_t)workspace & (kAlign - 1))) return set_err(nullptr, TPCCA_E_ARG, "workspace must be a 256-byte aligned device pointer");
  if (workspace_bytes < L.total)
    return set_err(nullptr, TPCCA_E_WORKSPACE, "workspace too small: %zu bytes given, %zu required", workspace_bytes, L.total);

  tpcca_ctx* c = new tpcca_ctx;
  c->device = cuda_device;
  c->sm_count = prop.multiProcessorCount > 0 ? prop.multiProcessorCount : 148;
  c->stream = (cudaStream_t)cuda_stream;
  c->ws = (char*)workspace;
  c->ws_bytes = workspace_bytes;
  c->N = N; c->CS = CS; c->ns = p->n_sectors; c->nr = p->n_rows; c->nb = bins_per_sector(p);
  c->L = L;
  c->sec.resize(c->ns);
  DevTables& t = c->tab;
  memset(&t, 0, sizeof t);
  t.n_rows = p->n_rows; t.n_sectors = p->n_sectors; t.bins_per_sector = (int32_t)c->nb;
  t.tc_max_gap = p->tc_max_gap; t.tc_min_hits = p->tc_min_hits; t.sel_permille = p->sel_max_shared_permille; t.res_inv_q = p->res_inv_quantum;
  {
    MgParams& m = c->mgp;
    m.per_side = p->sectors_per_side; m.max_row_gap = p->mg_max_row_gap; m.ca = p->sector_cos; m.sa = p->sector_sin;
    m.dy = p->mg_dy; m.dz = p->mg_dz; m.ds = p->mg_dsin; m.zpre = p->mg_zpre;
    m.n_zb = (int32_t)mg_z_buckets(p, &m.zb_lo, &m.zb_inv);
  }
  t.grid_z_lo = p->grid_z_lo; t.Bc = p->kappa_per_qpt; t.err2_y = p->err2_y; t.err2_z = p->err2_z;
  for (int i = 0; i < 5; ++i) t.init_cov[i] = p->init_cov[i];
  t.win_y = p->tc_win_y; t.win_z = p->tc_win_z; t.gate = p->tc_gate; t.max_sinphi = p->max_sinphi;
  t.margin = p->grid_margin;
  int32_t base = 0;
  for (int r = 0; r < p->n_rows; ++r) {
    t.row_x[r] = p->row_x[r]; t.y_lo[r] = p->grid_y_lo[r]; t.inv_by[r] = p->grid_inv_bin_y[r];
    t.inv_bz[r] = p->grid_inv_bin_z[r]; t.ny[r] = p->grid_ny[r]; t.nz[r] = p->grid_nz[r];
    t.ny_hi[r] = (float)(p->grid_ny[r] - 1); t.nz_hi[r] = (float)(p->grid_nz[r] - 1);
    t.bin_base[r] = base; base += p->grid_ny[r] * p->grid_nz[r];
    t.hy_up[r] = p->nf_hy_up[r]; t.hz_up[r] = p->nf_hz_up[r]; t.hy_dn[r] = p->nf_hy_dn[r];
    t.hz_dn[r] = p->nf_hz_dn[r]; t.nf_cut[r] = p->nf_cut[r];
  }
  t.bin_base[p->n_rows] = base;
  {
    int32_t cb = 0;
    const int kSlab = 1 << slab_shift_for(p, c->N);
    t.slab_shift = slab_shift_for(p, c->N);
    for (int r = 0; r < p->n_rows; ++r) { t.cb_base[r] = cb; cb += (p->grid_nz[r] + kSlab - 1) / kSlab; }
    t.cb_base[p->n_rows] = cb;
    t.n_cb = cb;
  }
  // S2 per-row constants; every float below is one fp32 operation on table values
  for (int r = 1; r + 1 < p->n_rows; ++r) {
    NfConst& k = t.nf[r];
    const float m = p->grid_margin;
    k.dA = make_float4(t.hy_dn[r], t.hz_dn[r], t.hy_dn[r] + m, t.hz_dn[r] + m);
    k.dB = make_float4(t.y_lo[r - 1], t.inv_by[r - 1], t.inv_bz[r - 1], t.grid_z_lo);
    k.dC = make_int4(t.ny[r - 1] - 1, t.nz[r - 1] - 1, t.ny[r - 1], t.bin_base[r - 1]);
    k.uA = make_float4(t.hy_up[r], t.hz_up[r], t.hy_up[r] + m, t.hz_up[r] + m);
    k.uB = make_float4(t.y_lo[r + 1], t.inv_by[r + 1], t.inv_bz[r + 1], t.grid_z_lo);
    k.uC = make_int4(t.ny[r + 1] - 1, t.nz[r + 1] - 1, t.ny[r + 1], t.bin_base[r + 1]);
    k.g = make_float4(t.row_x[r + 1] - t.row_x[r], t.row_x[r] - t.row_x[r - 1], t.nf_cut[r], 0.0f);
  }
  for (int r = 0; r < kMaxRows; ++r) c->nftab.row[r] = t.nf[r];
  {
    // S5 processing order: coarse buckets of a sector by ascending lower z edge, then row
    std::vector<std::pair<std::pair<float, int>, int>> zo;
    for (int r = 0; r < p->n_rows; ++r)
      for (int k = 0; k < t.cb_base[r + 1] - t.cb_base[r]; ++k)
        zo.push_back({{(float)(k << t.slab_shift) / p->grid_inv_bin_z[r], r}, t.cb_base[r] + k});
    std::sort(zo.begin(), zo.end());
    std::vector<int32_t> zl(2 * zo.size());
    for (size_t i = 0; i < zo.size(); ++i) zl[i] = zo[i].second;
    for (int r = 0; r < p->n_rows; ++r)      // second half: coarse bucket -> (row, slab), read by k_grid_sort
      for (int k = 0; k < t.cb_base[r + 1] - t.cb_base[r]; ++k) zl[zo.size() + (size_t)(t.cb_base[r] + k)] = r | (k << 8);
    cudaError_t ez = cudaMemcpyAsync(c->at<int32_t>(L.zorder), zl.data(), 4 * zl.size(), cudaMemcpyHostToDevice, c->stream);
    if (ez == cudaSuccess) ez = cudaStreamSynchronize(c->stream);
    if (ez != cudaSuccess) {
      set_err(nullptr, TPCCA_E_CUDA, "tpcca_create: %s", cudaGetErrorString(ez));
      tpcca_destroy(c);      // one cleanup path: releases whatever the partially built context owns
      return TPCCA_E_CUDA;
    }
  }
  cudaError_t e1 = cudaMemcpyAsync(c->at<DevTables>(L.tables), &t, sizeof t, cudaMemcpyHostToDevice, c->stream);
  if (e1 == cudaSuccess) e1 = cudaStreamSynchronize(c->stream);
  if (e1 == cudaSuccess) e1 = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
  for (int k = 0; k < tpcca_ctx::kRing && e1 == cudaSuccess; ++k)
    for (int i = 0; i < 9 && e1 == cudaSuccess; ++i) e1 = cudaEventCreate(&c->ev[k][i]);
  if (e1 != cudaSuccess) {
    set_err(nullptr, TPCCA_E_CUDA, "tpcca_create: %s", cudaGetErrorString(e1));
    tpcca_destroy(c);
    return TPCCA_E_CUDA;
  }
  {
    int occ = 0;
    // S2 kernel instance: the hit cache holds kNfK hits per side (5 blocks per SM) or, for dense time frames (more
    // than ~0.7 clusters per grid bin at the context's capacity: windows with more than kNfK hits are common there
    // and each one stalls its warp in the uncached path), kNfKDense hits (4 blocks per SM)
    c->nf_dense = (double)c->N > 0.7 * (double)c->ns * (double)c->nb;
    const void* nf_fn = c->nf_dense ? (const void*)k_neighbours<kNfKDense> : (const void*)k_neighbours<kNfK>;
    const size_t nf_smem = c->nf_dense ? sizeof(NfSmem<kNfKDense>) : sizeof(NfSmem<kNfK>);
    cudaError_t e2 = cudaFuncSetAttribute(nf_fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)nf_smem);
    if (e2 != cudaSuccess) {
      set_err(nullptr, TPCCA_E_CUDA, "tpcca_create: shared memory opt-in of k_neighbours failed: %s", cudaGetErrorString(e2));
      tpcca_destroy(c);
      return TPCCA_E_CUDA;
    }
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, nf_fn, kNfThreads, nf_smem) == cudaSuccess && occ > 0)
      c->nf_blocks_per_sm = occ;
  }
  *out_ctx = c;
  return TPCCA_OK;
}

int tpcca_reset(tpcca_ctx* c) {
  if (!c) return TPCCA_E_ARG;
  for (auto& s : c->sec) s = tpcca_ctx::Sec();
  c->in_used = 0;
  c->done_mask = 0;
  c->desc_valid = false;
  c->status_valid = false;
  return TPCCA_OK;
}

int tpcca_load_clusters(tpcca_ctx* c, int sector, int64_t n, const float* x, const float* y, const float* z,
                        const float* charge, const uint16_t* row, int mem_space) {
  (void)x; (void)charge;   // part of the cluster record, not read by S1-S5 (tpcca.h)
  if (!c) return TPCCA_E_ARG;
  if (sector < 0 || sector >= c->ns) return set_err(c, TPCCA_E_ARG, "sector %d out of range", sector);
  if (n < 0 || (n > 0 && (!y || !z || !row))) return set_err(c, TPCCA_E_ARG, "n < 0 or y/z/row NULL");
  if (mem_space < 0 || mem_space > 2) return set_err(c, TPCCA_E_ARG, "bad mem_space");
  if (c->sec[sector].loaded) return set_err(c, TPCCA_E_STATE, "sector %d already loaded; call tpcca_reset first", sector);
  int64_t tot = n;
  for (auto& s : c->sec) if (s.loaded) tot += s.n;
  if (tot > c->N) return set_err(c, TPCCA_E_WORKSPACE, "%lld clusters exceed max_clusters_total %lld", (long long)tot, (long long)c->N);
  GUARD(c);
  auto& S = c->sec[sector];
  if (mem_space == TPCCA_MEM_DEVICE_BORROW || n == 0) {
    S.y = y; S.z = z; S.row = row;
  } else {
    // 8-element alignment keeps every sector's copy 16-byte aligned
    const int64_t o = c->in_used;
    float* dy = c->at<float>(c->L.in_y) + o;
    float* dz = c->at<float>(c->L.in_z) + o;
    uint16_t* dr = c->at<uint16_t>(c->L.in_row) + o;
    const cudaMemcpyKind k = mem_space == TPCCA_MEM_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    CU(c, cudaMemcpyAsync(dy, y, 4 * (size_t)n, k, c->stream));
    CU(c, cudaMemcpyAsync(dz, z, 4 * (size_t)n, k, c->stream));
    CU(c, cudaMemcpyAsync(dr, row, 2 * (size_t)n, k, c->stream));
    S.y = dy; S.z = dz; S.row = dr;
    c->in_used += (n + 7) / 8 * 8;   // (fits: the total check above bounds the sum of n by N)
  }
  S.n = n; S.loaded = true;
  c->done_mask = 0;
  c->desc_valid = false;
  c->status_valid = false;
  return TPCCA_OK;
}

int tpcca_run(tpcca_ctx* c, uint32_t mask) {
  if (!c) return TPCCA_E_ARG;
  mask &= (TPCCA_STAGE_ALL | TPCCA_STAGE_SELECT | TPCCA_STAGE_RESIDUALS | TPCCA_STAGE_MERGE);
  if (!mask) return set_err(c, TPCCA_E_ARG, "empty stage mask");
  // a stage needs everything before it
  for (int i = 0; i < 8; ++i)
    if (mask & (1u << i)) {
      const uint32_t need = (1u << i) - 1u;
      if ((need & ~(c->done_mask | mask)) != 0)
        return set_err(c, TPCCA_E_STATE, "stage %d needs the outputs of earlier stages (done 0x%x, asked 0x%x)", i + 1, c->done_mask, mask);
    }
  GUARD(c);
  const Layout& L = c->L;
  cudaStream_t st = c->stream;
  c->launches = 0;
  c->status_valid = false;
  // ---- sector descriptors
  if (!c->desc_valid) {
    c->desc.assign(kMaxSectors + 1, SectorDesc{});
    int64_t off = 0, t256 = 0, t2048 = 0;
    for (int s = 0; s <= c->ns; ++s) {
      SectorDesc& d = c->desc[s];
      const int64_t n = s < c->ns ? c->sec[s].n : 0;
      if (s < c->ns) { d.y = c->sec[s].y; d.z = c->sec[s].z; d.row = c->sec[s].row; }
      d.n = (int32_t)n; d.off = (int32_t)off; d.tile256 = (int32_t)t256; d.tile2048 = (int32_t)t2048;
      off += n; t256 += (n + 255) / 256; t2048 += (n + 2047) / 2048;
    }
    c->n_total = off; c->n_tiles256 = (int)t256; c->n_tiles2048 = (int)t2048;
    int64_t mx = 0;
    for (int s = 0; s < c->ns; ++s) mx = std::max<int64_t>(mx, (c->sec[s].n + 255) / 256);
    c->max_tiles256 = (int)mx;
    CU(c, cudaMemcpyAsync(c->at<SectorDesc>(L.sec), c->desc.data(), sizeof(SectorDesc) * (kMaxSectors + 1), cudaMemcpyHostToDevice, st));
    c->desc_valid = true;
  }
  const DevTables* T = c->at<DevTables>(L.tables);
  const SectorDesc* sec = c->at<SectorDesc>(L.sec);
  DevStatus* status = c->at<DevStatus>(L.status);
  int64_t* tot = c->at<int64_t>(L.tot);     // [8]: pairs of scan totals (S4: 0,1; S5: 2,3; S4 order: 4,5; S6: 6,7)
  float2* syz = c->at<float2>(L.syz);
  int32_t* order = c->at<int32_t>(L.order);
  uint32_t* bin_start = c->at<uint32_t>(L.bin_start);
  int32_t* row_start = c->at<int32_t>(L.row_start);
  int2* tile_cnt = c->at<int2>(L.tile_cnt);
  longlong2* tile_off = c->at<longlong2>(L.tile_off);
  int32_t* start_hit = c->at<int32_t>(L.start_hit);
  const int32_t cap = (int32_t)c->CS;
  const int slot_ev = (int)(c->run_count % tpcca_ctx::kRing);
  c->ev_mask[slot_ev] = 0;
  // end of a stage: its event, and the launch errors of ITS kernels (so a failed launch names its stage)
  static const char* const kStageName[9] = {"start", "S1 grid", "S2 neighbours", "S3 clean", "S4 start hits", "S5 tracklets", "S6 selector", "S7 residuals", "S8 merge"};
  cudaError_t stage_err = cudaSuccess;
  int stage_bad = -1;
  auto mark = [&](int i) {
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaEventRecord(c->ev[slot_ev][i], st);
    if (e != cudaSuccess && stage_err == cudaSuccess) { stage_err = e; stage_bad = i; }
  };
  mark(0);

  if (mask & TPCCA_STAGE_GRID) {
    // (zeroing is done by kernels, not cudaMemsetAsync: a memset may be queued on a copy engine, where it waits
    // for the kernels before it and blocks the copies of other contexts queued behind it)
    k_zero_words<<<1, 256, 0, st>>>(reinterpret_cast<uint32_t*>(status), sizeof(DevStatus) / 4);
    uint32_t* cb_cnt = c->at<uint32_t>(L.cb_cnt);
    uint32_t* cb_start = c->at<uint32_t>(L.cb_start);
    uint32_t* big = c->at<uint32_t>(L.big_list);
    GridRec* rec = c->at<GridRec>(L.rec);
    {
      const size_t nw = (size_t)c->ns * (size_t)(L.n_cb + 1);
      k_zero_words<<<(unsigned)std::min<size_t>((nw + 1023) / 1024, 1024), 256, 0, st>>>(cb_cnt, nw);
      c->launches += 2;
    }
    if (c->n_tiles256 > 0) {
      k_cb_count<<<(unsigned)(c->ns * c->max_tiles256), 256, 0, st>>>(T, sec, cb_cnt, reinterpret_cast<uint32_t*>(order), status);   // `order` is free until level 2
      ++c->launches;
    }
    k_cb_scan<<<c->ns, 1024, 0, st>>>(T, cb_cnt, cb_start);
    ++c->launches;
    if (c->n_tiles256 > 0) {
      k_cb_scatter<<<c->n_tiles256, 256, 0, st>>>(T, sec, cb_start, reinterpret_cast<const uint32_t*>(order), rec);
      ++c->launches;
    }
    k_grid_sort<<<(unsigned)(c->ns * L.n_cb), 256, 0, st>>>(T, sec, c->at<int32_t>(L.zorder) + L.n_cb, cb_start, rec, syz, order, bin_start, big, status);
    k_grid_big<<<c->sm_count * 4, 256, 0, st>>>(T, sec, cb_start, rec, syz, order, bin_start, big, status);
    c->launches += 2;
    k_row_tables<<<1, 1024, 0, st>>>(T, bin_start, row_start, c->at<int32_t>(L.nf_tile_start), status);
    c->launches += 1;
  }
  mark(1);
  if ((mask & TPCCA_STAGE_NEIGHBOURS) && c->n_tiles256 > 0) {
    const int64_t tiles_ub = c->n_total / kNfTile + (int64_t)c->ns * c->nr;
    const int grid = (int)std::min<int64_t>(tiles_ub, (int64_t)c->sm_count * c->nf_blocks_per_sm);
    NfTileDesc* nfd = c->at<NfTileDesc>(L.nf_desc);
    const int32_t* nf_ts = c->at<int32_t>(L.nf_tile_start);
    k_nf_plan<<<std::min(c->ns * c->nr, c->sm_count * 64), 128, 0, st>>>(T, sec, syz, bin_start, row_start, nf_ts, nfd);
    if (c->nf_dense)
      k_neighbours<kNfKDense><<<grid, kNfThreads, sizeof(NfSmem<kNfKDense>), st>>>(c->nftab, syz, bin_start, order, (uint32_t)(c->nb + 1),
                                                                                   nf_ts + (size_t)c->ns * c->nr, nfd, c->at<int32_t>(L.up_raw),
                                                                                   c->at<int32_t>(L.dn_raw));
    else
      k_neighbours<kNfK><<<grid, kNfThreads, sizeof(NfSmem<kNfK>), st>>>(c->nftab, syz, bin_start, order, (uint32_t)(c->nb + 1),
                                                                         nf_ts + (size_t)c->ns * c->nr, nfd, c->at<int32_t>(L.up_raw),
                                                                         c->at<int32_t>(L.dn_raw));
    c->launches += 2;
  }
  mark(2);
  if ((mask & TPCCA_STAGE_CLEAN) && c->n_tiles2048 > 0) {
    k_clean_links<<<c->n_tiles2048, 256, 0, st>>>(T, sec, c->at<int32_t>(L.up_raw), c->at<int32_t>(L.dn_raw),
                                                 c->at<int32_t>(L.up), c->at<int32_t>(L.dn), tile_cnt, c->at<uint32_t>(L.start_bits), status);
    ++c->launches;
  }
  mark(3);
  if (mask & TPCCA_STAGE_START) {
    // tile_cnt is S3's by-product; if S3 ran in an earlier call S5's scans may have reused the
    // buffer, so S4 on its own recounts through S3's kernel (cheap, idempotent).
    if (!(mask & TPCCA_STAGE_CLEAN) && c->n_tiles2048 > 0) {
      k_clean_links<<<c->n_tiles2048, 256, 0, st>>>(T, sec, c->at<int32_t>(L.up_raw), c->at<int32_t>(L.dn_raw),
                                                   c->at<int32_t>(L.up), c->at<int32_t>(L.dn), tile_cnt, c->at<uint32_t>(L.start_bits), status);
      ++c->launches;
    }
    k_scan_pairs<<<1, 1024, 0, st>>>(tile_cnt, tile_off, c->n_tiles2048, tot);
    k_start_offsets<<<1, kMaxSectors + 1, 0, st>>>(T, sec, tile_off, tot, c->n_tiles2048, cap, status);
    c->launches += 2;
    if (c->n_tiles2048 > 0) {
      k_start_hits<<<c->n_tiles2048, 256, 0, st>>>(T, sec, c->at<uint32_t>(L.start_bits), tile_off, cap, start_hit);
      ++c->launches;
    }
    {   // processing order of S5: start-hit slots by (sector, z)
      const int nbk = (int)(c->ns * L.n_cb), nblk = (nbk + 255) / 256;
      int32_t* shc = c->at<int32_t>(L.sh_cnt);
      int2* blc = c->at<int2>(L.sh_blk);
      longlong2* shp = c->at<longlong2>(L.sh_pre);
      k_sh_bucket_counts<<<nblk, 256, 0, st>>>(T, status, c->at<int32_t>(L.zorder), c->at<uint32_t>(L.cb_start), start_hit, cap,
                                               c->at<int32_t>(L.sh_first), shc, blc);
      k_scan_pairs<<<1, 1024, 0, st>>>(blc, shp, nblk, tot + 4);
      k_sh_perm<<<nblk, 256, 0, st>>>(T, c->at<int32_t>(L.zorder), start_hit, c->at<int32_t>(L.sh_first), shc, shp, c->at<int4>(L.perm));
      c->launches += 3;
    }
  }
  mark(4);
  if (mask & TPCCA_STAGE_TRACKLETS) {
    TrackOut o;
    o.x_ref = c->at<float>(L.o_x_ref); o.z_ref = c->at<float>(L.o_z_ref); o.par = c->at<float>(L.o_par);
    o.cov = c->at<float>(L.o_cov); o.chi2 = c->at<float>(L.o_chi2); o.n_hits = c->at<int32_t>(L.o_n_hits);
    o.n_fit = c->at<int32_t>(L.o_n_fit); o.first_row = c->at<int32_t>(L.o_first); o.last_row = c->at<int32_t>(L.o_last);
    o.start_hit = c->at<int32_t>(L.o_start); o.hit_offset = c->at<int32_t>(L.o_hit_offset); o.hit_idx = c->at<int32_t>(L.o_hit_idx);
    int32_t* hits = c->at<int32_t>(L.hits);
    float4* trk_f = c->at<float4>(L.trk_v);
    int32_t* trk_i = c->at<int32_t>(L.trk_n);
    const int cap_tiles = (int)((c->CS + 1023) / 1024);
    static_assert(sizeof(status->work_counter) % 4 == 0 && sizeof(status->work) % 4 == 0, "word-sized counters");
    k_zero_words<<<1, 32, 0, st>>>(reinterpret_cast<uint32_t*>(status->work_counter), sizeof(status->work_counter) / 4);
    k_zero_words<<<1, 32, 0, st>>>(reinterpret_cast<uint32_t*>(status->work), sizeof(status->work) / 4);
    c->launches += 2;
    const DevTables& t = c->tab;
    S5Params sp;
    sp.Bc = t.Bc; sp.err2_y = t.err2_y; sp.err2_z = t.err2_z; sp.max_sinphi = t.max_sinphi;
    sp.ic0 = t.init_cov[0]; sp.ic1 = t.init_cov[1]; sp.ic2 = t.init_cov[2]; sp.ic3 = t.init_cov[3]; sp.ic4 = t.init_cov[4];
    sp.win_y = t.win_y; sp.win_z = t.win_z; sp.gate = t.gate; sp.margin = t.margin; sp.grid_z_lo = t.grid_z_lo;
    sp.n_rows = t.n_rows; sp.n_sectors = t.n_sectors; sp.max_gap = t.tc_max_gap; sp.min_hits = t.tc_min_hits;
    sp.bins_per_sector = t.bins_per_sector;
    float4* hs_f = c->at<float4>(L.hs);
    const int4* perm = c->at<int4>(L.perm);
    k_tracklets<MODE_A><<<c->sm_count * kS5BlocksPerSMA, kS5Threads, 0, st>>>(T, sec, status, sp, syz, bin_start, order, c->at<int32_t>(L.up),
                                                                              perm, cap, hits, trk_f, trk_i, hs_f);
    k_tracklets<MODE_B><<<c->sm_count * kS5BlocksPerSM, kS5Threads, 0, st>>>(T, sec, status, sp, syz, bin_start, order, c->at<int32_t>(L.up),
                                                                              perm, cap, hits, trk_f, trk_i, hs_f);
    k_tracklets<MODE_C1><<<c->sm_count * kS5BlocksPerSM, kS5Threads, 0, st>>>(T, sec, status, sp, syz, bin_start, order, c->at<int32_t>(L.up),
                                                                              perm, cap, hits, trk_f, trk_i, hs_f);
    k_tracklets<MODE_C2><<<c->sm_count * kS5BlocksPerSM, kS5Threads, 0, st>>>(T, sec, status, sp, syz, bin_start, order, c->at<int32_t>(L.up),
                                                                              perm, cap, hits, trk_f, trk_i, hs_f);
    k_track_tile_sums<<<cap_tiles, 1024, 0, st>>>(status, trk_i, tile_cnt);
    k_scan_pairs<<<1, 1024, 0, st>>>(tile_cnt, tile_off, cap_tiles, tot + 2);
    k_track_sector_bases<<<1, kMaxSectors + 1, 0, st>>>(T, status, trk_i, tile_off, tot + 2);
    k_track_gather<<<cap_tiles, 1024, 0, st>>>(T, status, start_hit, cap, hits, trk_f, trk_i, tile_off, o, c->at<int32_t>(L.slot_trk));
    k_track_close_empty<<<1, kMaxSectors, 0, st>>>(T, status, o);
    c->launches += 9;
  }
  mark(5);
  if (mask & TPCCA_STAGE_SELECT) {
    // S6 buffers: own_key / owner live in the S1 level-1 record buffer (free after S1), the compact table of the
    // selected tracks in the S5 scratch (slot records, parked tracklets, per-tracklet hit lines: free after S5)
    TrackOut in;
    in.x_ref = c->at<float>(L.o_x_ref); in.z_ref = c->at<float>(L.o_z_ref); in.par = c->at<float>(L.o_par);
    in.cov = c->at<float>(L.o_cov); in.chi2 = c->at<float>(L.o_chi2); in.n_hits = c->at<int32_t>(L.o_n_hits);
    in.n_fit = c->at<int32_t>(L.o_n_fit); in.first_row = c->at<int32_t>(L.o_first); in.last_row = c->at<int32_t>(L.o_last);
    in.start_hit = c->at<int32_t>(L.o_start); in.hit_offset = c->at<int32_t>(L.o_hit_offset); in.hit_idx = c->at<int32_t>(L.o_hit_idx);
    SelOut so = sel_out(c);
    uint32_t* own_key = c->at<uint32_t>(L.rec);          // ownership keys, decoded in place to `owner` at the end
    int32_t* n_own = c->at<int32_t>(L.sel_n_own);
    const int32_t* slot_trk = c->at<int32_t>(L.slot_trk);
    const int4* perm = c->at<int4>(L.perm);
    const int cap_tiles = (int)((c->CS + 1023) / 1024);
    const size_t nk = (size_t)std::max<int64_t>(c->n_total, 1);
    k_zero_words<<<(unsigned)std::min<size_t>((nk + 1023) / 1024, (size_t)c->sm_count * 32), 256, 0, st>>>(own_key, nk);
    const int warp_grid = (int)std::min<int64_t>((c->CS + 7) / 8, (int64_t)c->sm_count * 8);
    k_sel_claim<<<warp_grid, 256, 0, st>>>(T, sec, status, perm, slot_trk, in.n_hits, in.hit_offset, in.hit_idx, own_key);
    k_sel_count<<<warp_grid, 256, 0, st>>>(T, sec, status, perm, slot_trk, in.n_hits, in.hit_offset, in.hit_idx, own_key, n_own);
    k_sel_tile_sums<<<cap_tiles, 1024, 0, st>>>(T, status, in.n_hits, n_own, tile_cnt);
    k_scan_pairs<<<1, 1024, 0, st>>>(tile_cnt, tile_off, cap_tiles, tot + 6);
    k_sel_sector_bases<<<1, kMaxSectors + 1, 0, st>>>(T, status, in.n_hits, n_own, tile_off, tot + 6);
    k_sel_gather<<<cap_tiles, 1024, 0, st>>>(T, status, cap, n_own, tile_off, in, so);
    k_sel_close_empty<<<1, kMaxSectors, 0, st>>>(T, status, so);
    k_sel_owner<<<(unsigned)std::min<size_t>((nk + 255) / 256, (size_t)c->sm_count * 32), 256, 0, st>>>(own_key, nk);
    c->launches += 9;
  }
  mark(6);
  if (mask & TPCCA_STAGE_RESIDUALS) {
    tpcca_residual* ro = c->at<tpcca_residual>(L.res);
    const size_t nk = (size_t)std::max<int64_t>(c->n_total, 1);
    k_res_init<<<(unsigned)std::min<size_t>((nk + 255) / 256, (size_t)c->sm_count * 32), 256, 0, st>>>(ro, nk);
    const MgBuf mb = mg_buf(c);
    k_residuals<<<(unsigned)((c->CS + 127) / 128), 128, 0, st>>>(T, sec, status, syz, row_start, c->at<int32_t>(L.rec), sel_out(c), cap, ro,
                                                                 mb.out_x, mb.out_p, mb.out_ok);
    c->launches += 2;
  }
  mark(7);
  if (mask & TPCCA_STAGE_MERGE) {
    const MgBuf mb = mg_buf(c);
    const SelOut so = sel_out(c);
    const size_t nbk = (size_t)c->ns * c->nr * c->mgp.n_zb + 1;
    uint32_t* cursor = c->at<uint32_t>(L.mg_cur);
    const unsigned g256 = (unsigned)((c->CS + 255) / 256), g128 = (unsigned)((c->CS + 127) / 128);
    k_zero_words<<<(unsigned)std::min<size_t>((nbk + 1023) / 1024, (size_t)c->sm_count * 8), 256, 0, st>>>(mb.bk_cnt, nbk + 1);
    k_zero_words<<<(unsigned)std::min<size_t>((nbk + 1023) / 1024, (size_t)c->sm_count * 8), 256, 0, st>>>(cursor, nbk + 1);
    k_mg_count<<<g256, 256, 0, st>>>(T, status, so, cap, c->mgp, mb);
    k_mg_scan<<<c->ns, 1024, 0, st>>>(T, status, mb.bk_cnt, (int)((nbk - 1) / c->ns));
    k_mg_scatter<<<g256, 256, 0, st>>>(T, status, so, cap, c->mgp, mb, cursor);
    k_mg_match<<<g128, 128, 0, st>>>(T, status, so, cap, c->mgp, mb);
    k_mg_link<<<g256, 256, 0, st>>>(T, status, mb);
    // chain heads, compacted: bk_list is free once the matching is done; the cursor array's last word counts them
    int32_t* head_list = mb.bk_list;
    uint32_t* n_heads = cursor + nbk;
    k_mg_heads<<<g256, 256, 0, st>>>(T, status, mb, head_list, n_heads);
    k_mg_refit<<<g128, 128, 0, st>>>(T, sec, status, syz, row_start, so, cap, c->mgp, mb, head_list, n_heads);
    c->launches += 9;
  }
  mark(8);
  if (stage_err != cudaSuccess)
    return set_err(c, TPCCA_E_CUDA, "tpcca_run: stage %s failed: %s", kStageName[stage_bad], cudaGetErrorString(stage_err));
  c->ev_mask[slot_ev] = mask;
  ++c->run_count;
  // S6's outputs alias S1 / S5 scratch: re-running either without S6 leaves no valid selection
  if ((mask & (TPCCA_STAGE_GRID | TPCCA_STAGE_TRACKLETS)) && !(mask & TPCCA_STAGE_SELECT)) c->done_mask &= ~(TPCCA_STAGE_SELECT | TPCCA_STAGE_RESIDUALS | TPCCA_STAGE_MERGE);
  if ((mask & TPCCA_STAGE_SELECT) && !(mask & TPCCA_STAGE_RESIDUALS)) c->done_mask &= ~(TPCCA_STAGE_RESIDUALS | TPCCA_STAGE_MERGE);
  if ((mask & (TPCCA_STAGE_GRID | TPCCA_STAGE_TRACKLETS | TPCCA_STAGE_RESIDUALS)) && !(mask & TPCCA_STAGE_MERGE)) c->done_mask &= ~TPCCA_STAGE_MERGE;
  c->done_mask |= mask;
  return TPCCA_OK;
}

int tpcca_sync(tpcca_ctx* c) {
  if (!c) return TPCCA_E_ARG;
  GUARD(c);
  return fetch_status(c);
}

int tpcca_get_counts(tpcca_ctx* c, int64_t out[7]) {
  if (!c || !out) return TPCCA_E_ARG;
  GUARD(c);
  int rc = fetch_status(c);
  if (rc) return rc;
  out[0] = c->n_total;
  out[1] = (c->done_mask & TPCCA_STAGE_START) ? c->status.n_start : 0;
  out[2] = (c->done_mask & TPCCA_STAGE_TRACKLETS) ? c->status.trk_off[c->ns] : 0;
  out[3] = (c->done_mask & TPCCA_STAGE_TRACKLETS) ? c->status.hit_off[c->ns] : 0;
  out[4] = c->nb;
  out[5] = (c->done_mask & TPCCA_STAGE_SELECT) ? c->status.sel_off[c->ns] : 0;
  out[6] = (c->done_mask & TPCCA_STAGE_SELECT) ? c->status.sel_hit_off[c->ns] : 0;
  return TPCCA_OK;
}

int tpcca_get_timings(tpcca_ctx* c, int runs_back, float ms[9]) {
  if (!c || !ms) return TPCCA_E_ARG;
  if (runs_back < 0 || runs_back >= tpcca_ctx::kRing) return set_err(c, TPCCA_E_ARG, "runs_back must be in 0..15");
  for (int i = 0; i < 9; ++i) ms[i] = 0.f;
  if (runs_back >= c->run_count) return set_err(c, TPCCA_E_STATE, "no such run");
  const int k = (int)((c->run_count - 1 - runs_back) % tpcca_ctx::kRing);
  if (!c->ev_mask[k]) return set_err(c, TPCCA_E_STATE, "no such run");
  GUARD(c);
  CU(c, cudaStreamSynchronize(c->stream));
  for (int i = 0; i < 5; ++i) CU(c, cudaEventElapsedTime(&ms[i], c->ev[k][i], c->ev[k][i + 1]));
  CU(c, cudaEventElapsedTime(&ms[5], c->ev[k][0], c->ev[k][5]));
  CU(c, cudaEventElapsedTime(&ms[6], c->ev[k][5], c->ev[k][6]));
  CU(c, cudaEventElapsedTime(&ms[7], c->ev[k][6], c->ev[k][7]));
  CU(c, cudaEventElapsedTime(&ms[8], c->ev[k][7], c->ev[k][8]));
  // the events around a stage are recorded whether or not the stage ran: a stage outside the run's mask would show
  // the few microseconds between two records.  The header promises 0 for it.
  const uint32_t m = c->ev_mask[k];
  for (int i = 0; i < 5; ++i) if (!(m & (1u << i))) ms[i] = 0.f;
  for (int i = 6; i < 9; ++i) if (!(m & (1u << (i - 1)))) ms[i] = 0.f;
  return TPCCA_OK;
}

int tpcca_get_work_counters(tpcca_ctx* c, int64_t out[5]) {
  if (!c || !out) return TPCCA_E_ARG;
  GUARD(c);
  int rc = fetch_status(c);
  if (rc) return rc;
  for (int i = 0; i < 5; ++i) out[i] = (int64_t)c->status.work[i];
  return TPCCA_OK;
}

int tpcca_get_info(const tpcca_ctx* c, int64_t out[8]) {
  if (!c || !out) return TPCCA_E_ARG;
  out[0] = c->tab.slab_shift; out[1] = c->tab.n_cb; out[2] = c->nf_dense ? kNfKDense : kNfK; out[3] = c->sm_count;
  out[4] = c->nf_blocks_per_sm; out[5] = c->N; out[6] = c->CS; out[7] = (int64_t)c->L.total;
  return TPCCA_OK;
}

int tpcca_get_launch_count(const tpcca_ctx* c, int64_t* out) {
  if (!c || !out) return TPCCA_E_ARG;
  *out = c->launches;
  return TPCCA_OK;
}

// Outputs of sectors [sec0, sec1) into views[0 .. sec1 - sec0): DEVICE pointers, or HOST copies into ONE pinned arena
// followed by one synchronise of the copy stream.
static int get_tracks_range(tpcca_ctx* c, int sec0, int sec1, int mem_space, uint32_t what, tpcca_tracks_view* views) {
  if (!c || !views) return TPCCA_E_ARG;
  if (sec0 < 0 || sec1 > c->ns || sec0 >= sec1) return set_err(c, TPCCA_E_ARG, "sector range %d..%d out of range", sec0, sec1);
  if (mem_space != TPCCA_MEM_HOST && mem_space != TPCCA_MEM_DEVICE) return set_err(c, TPCCA_E_ARG, "bad mem_space");
  if (!c->done_mask || !c->desc_valid) return set_err(c, TPCCA_E_STATE, "nothing was run");
  GUARD(c);
  const bool host = mem_space == TPCCA_MEM_HOST;
  // HOST copies wait only for the last stage whose outputs are asked for (so that the links of a time
  // frame can travel while S5 still runs); the track counts are filled once S5 is covered.
  int need_stage = 1;
  if (what & TPCCA_OUT_LINKS_RAW) need_stage = 2;
  if (what & TPCCA_OUT_LINKS) need_stage = 3;
  if (what & TPCCA_OUT_START) need_stage = 4;
  if (what & TPCCA_OUT_TRACKS) need_stage = 5;
  if ((what & (TPCCA_OUT_SELECTION | TPCCA_OUT_TRACKS_SEL)) && (c->done_mask & TPCCA_STAGE_SELECT)) need_stage = 6;
  if ((what & TPCCA_OUT_RESIDUALS) && (c->done_mask & TPCCA_STAGE_RESIDUALS)) need_stage = 7;
  if ((what & TPCCA_OUT_MERGE) && (c->done_mask & TPCCA_STAGE_MERGE)) need_stage = 8;
  if ((what & TPCCA_OUT_TRACKS) && (what & TPCCA_OUT_TRACKS_SEL))
    return set_err(c, TPCCA_E_ARG, "TPCCA_OUT_TRACKS and TPCCA_OUT_TRACKS_SEL fill the same fields: ask for one");
  while (need_stage > 1 && need_stage <= 5 && !(c->done_mask & (1u << (need_stage - 1)))) --need_stage;     // stages that were never run deliver nothing
  const bool partial = host && need_stage < 5 && (c->done_mask & TPCCA_STAGE_TRACKLETS) && c->run_count > 0;
  int rc = partial ? fetch_status_after(c, std::max(need_stage, (c->done_mask & TPCCA_STAGE_START) ? 4 : need_stage)) : fetch_status(c);
  if (rc) return rc;
  const Layout& L = c->L;
  const DevStatus& S = c->status;
  // the arrays to deliver: (destination field, device source, bytes); par / cov are strided planes
  struct Item { const void** dst; const void* src; size_t bytes; int planes; };
  std::vector<Item> items;
  auto add = [&](const void* const* dst, const void* src, size_t bytes, int planes = 1) {
    items.push_back(Item{(const void**)dst, src, bytes, planes});
  };
  for (int sector = sec0; sector < sec1; ++sector) {
  tpcca_tracks_view* v = views + (sector - sec0);
  memset(v, 0, sizeof *v);
  const int64_t n = c->desc[sector].n, off = c->desc[sector].off;
  const uint32_t done = partial ? (c->done_mask & ~(TPCCA_STAGE_TRACKLETS | TPCCA_STAGE_SELECT | TPCCA_STAGE_RESIDUALS | TPCCA_STAGE_MERGE)) : c->done_mask;
  v->n_clusters = n;
  v->n_bins = c->nb;
  int64_t s0 = 0, s1 = 0, t0 = 0, nt = 0, h0 = 0, h1 = 0;
  if (done & TPCCA_STAGE_START) { s0 = S.start_off[sector]; s1 = S.start_off[sector + 1]; v->n_start = s1 - s0; }
  if (done & TPCCA_STAGE_TRACKLETS) {
    t0 = S.trk_off[sector]; nt = S.trk_off[sector + 1] - t0; h0 = S.hit_off[sector]; h1 = S.hit_off[sector + 1];
    v->n_tracks = nt; v->n_hits = h1 - h0;
  }
  if ((what & TPCCA_OUT_ORDER) && (done & TPCCA_STAGE_GRID))
    add((const void* const*)&v->order, c->at<int32_t>(L.order) + off, 4 * (size_t)n);
  if ((what & TPCCA_OUT_GRID) && (done & TPCCA_STAGE_GRID)) {
    add((const void* const*)&v->syz, c->at<float2>(L.syz) + off, 8 * (size_t)n);
    add((const void* const*)&v->bin_start, c->at<uint32_t>(L.bin_start) + (size_t)sector * (c->nb + 1), 4 * (size_t)(c->nb + 1));
    add((const void* const*)&v->row_start, c->at<int32_t>(L.row_start) + (size_t)sector * (c->nr + 1), 4 * (size_t)(c->nr + 1));
  }
  if ((what & TPCCA_OUT_LINKS_RAW) && (done & TPCCA_STAGE_NEIGHBOURS)) {
    add((const void* const*)&v->link_up_raw, c->at<int32_t>(L.up_raw) + off, 4 * (size_t)n);
    add((const void* const*)&v->link_dn_raw, c->at<int32_t>(L.dn_raw) + off, 4 * (size_t)n);
  }
  if ((what & TPCCA_OUT_LINKS) && (done & TPCCA_STAGE_CLEAN)) {
    add((const void* const*)&v->link_up, c->at<int32_t>(L.up) + off, 4 * (size_t)n);
    add((const void* const*)&v->link_dn, c->at<int32_t>(L.dn) + off, 4 * (size_t)n);
  }
  if ((what & TPCCA_OUT_START) && (done & TPCCA_STAGE_START))
    add((const void* const*)&v->start_hit, c->at<int32_t>(L.start_hit) + s0, 4 * (size_t)(s1 - s0));
  if ((what & TPCCA_OUT_TRACKS) && (done & TPCCA_STAGE_TRACKLETS)) {
    add((const void* const*)&v->x_ref, c->at<float>(L.o_x_ref) + t0, 4 * (size_t)nt);
    add((const void* const*)&v->z_ref, c->at<float>(L.o_z_ref) + t0, 4 * (size_t)nt);
    add((const void* const*)&v->chi2, c->at<float>(L.o_chi2) + t0, 4 * (size_t)nt);
    add((const void* const*)&v->par, c->at<float>(L.o_par) + t0, 4 * (size_t)nt, 5);
    add((const void* const*)&v->cov, c->at<float>(L.o_cov) + t0, 4 * (size_t)nt, 15);
    add((const void* const*)&v->n_hits_trk, c->at<int32_t>(L.o_n_hits) + t0, 4 * (size_t)nt);
    add((const void* const*)&v->n_fit, c->at<int32_t>(L.o_n_fit) + t0, 4 * (size_t)nt);
    add((const void* const*)&v->first_row, c->at<int32_t>(L.o_first) + t0, 4 * (size_t)nt);
    add((const void* const*)&v->last_row, c->at<int32_t>(L.o_last) + t0, 4 * (size_t)nt);
    add((const void* const*)&v->trk_start_hit, c->at<int32_t>(L.o_start) + t0, 4 * (size_t)nt);
    add((const void* const*)&v->hit_offset, c->at<int32_t>(L.o_hit_offset) + t0 + sector, 4 * (size_t)(nt + 1));
    add((const void* const*)&v->hit_idx, c->at<int32_t>(L.o_hit_idx) + h0, 4 * (size_t)(h1 - h0));
    v->trk_stride = host ? nt : c->CS;
  }
  if (done & TPCCA_STAGE_SELECT) {
    const int64_t k0 = S.sel_off[sector], nk = S.sel_off[sector + 1] - k0;
    const int64_t g0 = S.sel_hit_off[sector], g1 = S.sel_hit_off[sector + 1];
    v->n_selected = nk; v->n_sel_hits = g1 - g0;
    if (what & TPCCA_OUT_SELECTION) {
      add((const void* const*)&v->owner, c->at<int32_t>(L.rec) + off, 4 * (size_t)n);
      add((const void* const*)&v->n_own, c->at<int32_t>(L.sel_n_own) + t0, 4 * (size_t)nt);
      add((const void* const*)&v->sel_track, c->at<int32_t>(L.sel_track) + k0, 4 * (size_t)nk);
    }
    if (what & TPCCA_OUT_TRACKS_SEL) {       // the S5 fields of the view, filled from the compact table of the selected tracks
      const SelOut so = sel_out(c);
      add((const void* const*)&v->x_ref, so.o.x_ref + k0, 4 * (size_t)nk);
      add((const void* const*)&v->z_ref, so.o.z_ref + k0, 4 * (size_t)nk);
      add((const void* const*)&v->chi2, so.o.chi2 + k0, 4 * (size_t)nk);
      add((const void* const*)&v->par, so.o.par + k0, 4 * (size_t)nk, 5);
      add((const void* const*)&v->cov, so.o.cov + k0, 4 * (size_t)nk, 15);
      add((const void* const*)&v->n_hits_trk, so.o.n_hits + k0, 4 * (size_t)nk);
      add((const void* const*)&v->n_fit, so.o.n_fit + k0, 4 * (size_t)nk);
      add((const void* const*)&v->first_row, so.o.first_row + k0, 4 * (size_t)nk);
      add((const void* const*)&v->last_row, so.o.last_row + k0, 4 * (size_t)nk);
      add((const void* const*)&v->trk_start_hit, so.o.start_hit + k0, 4 * (size_t)nk);
      add((const void* const*)&v->hit_offset, so.o.hit_offset + k0 + sector, 4 * (size_t)(nk + 1));
      add((const void* const*)&v->hit_idx, so.o.hit_idx + g0, 4 * (size_t)(g1 - g0));
      v->trk_stride = host ? nk : c->CS;
    }
  }
  if ((done & TPCCA_STAGE_RESIDUALS) && (what & TPCCA_OUT_RESIDUALS)) {
    add((const void* const*)&v->res, c->at<tpcca_residual>(L.res) + off, sizeof(tpcca_residual) * (size_t)n);
  }
  if ((done & TPCCA_STAGE_MERGE) && (what & TPCCA_OUT_MERGE)) {
    const MgBuf mb = mg_buf(c);
    const int64_t k0 = S.sel_off[sector], nk = S.sel_off[sector + 1] - k0;
    const size_t by = 4 * (size_t)nk;
    add((const void* const*)&v->mg_next_sec, mb.next_sec + k0, by); add((const void* const*)&v->mg_next_trk, mb.next_trk + k0, by);
    add((const void* const*)&v->mg_prev_sec, mb.prev_sec + k0, by); add((const void* const*)&v->mg_prev_trk, mb.prev_trk + k0, by);
    add((const void* const*)&v->mg_n_seg, mb.n_seg + k0, by); add((const void* const*)&v->mg_n_hits, mb.n_hits + k0, by);
    add((const void* const*)&v->mg_n_fit, mb.n_fit + k0, by); add((const void* const*)&v->mg_first_row, mb.first_row + k0, by);
    add((const void* const*)&v->mg_last_row, mb.last_row + k0, by); add((const void* const*)&v->mg_frame_seg, mb.frame_seg + k0, by);
    add((const void* const*)&v->mg_x_ref, mb.x_ref + k0, by); add((const void* const*)&v->mg_z_ref, mb.z_ref + k0, by);
    add((const void* const*)&v->mg_chi2, mb.chi2 + k0, by);
    add((const void* const*)&v->mg_par, mb.par + k0, by, 5); add((const void* const*)&v->mg_cov, mb.cov + k0, by, 15);
    v->mg_stride = host ? nk : c->CS;
  }
  }   // sectors
  if (!host) {
    for (auto& it : items) *it.dst = it.src;
    return TPCCA_OK;
  }
  size_t need = 256;
  for (auto& it : items) need += align_up(it.bytes * it.planes + 4);
  if (need > c->arena_bytes) {
    if (c->arena) cudaFreeHost(c->arena);
    c->arena = nullptr; c->arena_bytes = 0;
    const size_t want = need + need / 4;
    cudaError_t e = cudaMallocHost((void**)&c->arena, want);
    if (e != cudaSuccess) return set_err(c, TPCCA_E_CUDA, "cudaMallocHost(%zu) failed: %s", want, cudaGetErrorString(e));
    c->arena_bytes = want;
  }
  // the copies run on the context's copy stream: it has already waited for the stage that made the
  // data (partial) or the whole run is complete (fetch_status synchronised the main stream)
  cudaStream_t cs = c->copy_stream;
  size_t cur = 0;
  for (auto& it : items) {
    char* dst = c->arena + cur;
    if (it.bytes) {
      // par / cov planes are CS elements apart on the device and packed (n_tracks apart) on the host: one copy per
      // plane (a 2-D copy would be bound by the device's maximum pitch, about 2 GiB, i.e. CS < 2^29)
      for (int pl = 0; pl < it.planes; ++pl)
        CU(c, cudaMemcpyAsync(dst + (size_t)pl * it.bytes, (const char*)it.src + (size_t)pl * 4 * (size_t)c->CS, it.bytes,
                              cudaMemcpyDeviceToHost, cs));
    }
    *it.dst = dst;
    cur += align_up(it.bytes * it.planes + 4);
  }
  CU(c, cudaStreamSynchronize(cs));
  return TPCCA_OK;
}

int tpcca_get_tracks(tpcca_ctx* c, int sector, int mem_space, uint32_t what, tpcca_tracks_view* v) {
  if (!c || !v) return TPCCA_E_ARG;
  if (sector < 0 || sector >= c->ns) return set_err(c, TPCCA_E_ARG, "sector %d out of range", sector);
  return get_tracks_range(c, sector, sector + 1, mem_space, what, v);
}

int tpcca_get_tracks_all(tpcca_ctx* c, int mem_space, uint32_t what, tpcca_tracks_view* views) {
  if (!c || !views) return TPCCA_E_ARG;
  return get_tracks_range(c, 0, c->ns, mem_space, what, views);
}

void tpcca_destroy(tpcca_ctx* c) {
  if (!c) return;
  DeviceGuard guard(c->device);
  cudaStreamSynchronize(c->stream);
  for (int k = 0; k < tpcca_ctx::kRing; ++k)
    for (int i = 0; i < 9; ++i) if (c->ev[k][i]) cudaEventDestroy(c->ev[k][i]);
  if (c->arena) cudaFreeHost(c->arena);
  if (c->copy_stream) { cudaStreamSynchronize(c->copy_stream); cudaStreamDestroy(c->copy_stream); }
  delete c;
}

}  // extern "C"

#include "tpcca_pipeline.cuh"
