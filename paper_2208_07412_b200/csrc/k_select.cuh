// S6 tracklet selector: per-cluster ownership by (n_hits, -track),
// tracklets that share too many of their hits are dropped, the survivors are gathered into a compact
// track table + hit CSR (the table a consumer downloads instead of the 4x larger clone-laden one).
#pragma once
#include "k_tracklets.cuh"

namespace tpcca {

// sector of global track t: largest s with trk_off[s] <= t (sectors without tracks are skipped)
__device__ __forceinline__ int sector_of_track(const DevStatus* __restrict__ st, int ns, int t) {
  int lo = 0, hi = ns - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (st->trk_off[mid] <= t) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// ownership key of track t_local with nh hits: larger = better; ties in nh -> the smaller track number wins.
// 32 bits: nh (<= TPCCA_MAX_ROWS = 256: 9 bits) | 0x7FFFFF - t_local (a sector with 2^23 or more tracks is refused:
// DevStatus::err_select).  0 = unclaimed (a real key has nh >= 1 in its top bits).
constexpr int kSelTrackBits = 23;
__device__ __forceinline__ uint32_t sel_key(int nh, int t_local) {
  return ((uint32_t)nh << kSelTrackBits) | (uint32_t)(((1 << kSelTrackBits) - 1) - t_local);
}

// Both passes walk the tracks in the PROCESSING ORDER of S5 (perm: sector by sector in ascending z), not in output
// order: the three or four clones of a particle then touch its ~100 clusters within a short time and the scattered
// 4-byte accesses hit L2 instead of DRAM.  slot_trk[slot] = global track of the start-hit slot (-1: rejected).
// ---- K6a: claim.  One warp per track: own_key[cluster] = max over the tracks holding it ---------------
__global__ void __launch_bounds__(256)
k_sel_claim(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, DevStatus* __restrict__ st,
            const int4* __restrict__ perm, const int32_t* __restrict__ slot_trk,
            const int32_t* __restrict__ n_hits, const int32_t* __restrict__ hit_offset, const int32_t* __restrict__ hit_idx,
            uint32_t* __restrict__ own_key) {
  if (st->err_capacity || st->err_range) return;
  const int n_start = st->n_start;
  const int lane = threadIdx.x & 31;
  for (int j = blockIdx.x * 8 + (threadIdx.x >> 5); j < n_start; j += gridDim.x * 8) {
    const int4 pr = __ldg(&perm[j]);
    const int t = slot_trk[pr.x];
    if (t < 0) continue;
    const int s = pr.y >> 16;
    const int t_local = t - st->trk_off[s];
    if (t_local >= (1 << kSelTrackBits) - 1) { if (lane == 0) st->err_select = 1; continue; }
    const int nh = n_hits[t];
    const long long h0 = st->hit_off[s] + hit_offset[t + s];
    const uint32_t key = sel_key(nh, t_local);
    uint32_t* ok = own_key + sec[s].off;
    for (int k = lane; k < nh; k += 32) {
      const int c = __ldcs(&hit_idx[h0 + k]);      // streamed once: keep L2 for the keys
      // (plain read first: most clusters are claimed by three or four clones and only the first few raise the key)
      if (ok[c] < key) atomicMax(&ok[c], key);
    }
  }
}

// ---- K6b: count.  One warp per track: n_own[t] = hits whose key is the track's own ----------------------
__global__ void __launch_bounds__(256)
k_sel_count(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, const DevStatus* __restrict__ st,
            const int4* __restrict__ perm, const int32_t* __restrict__ slot_trk,
            const int32_t* __restrict__ n_hits, const int32_t* __restrict__ hit_offset, const int32_t* __restrict__ hit_idx,
            const uint32_t* __restrict__ own_key, int32_t* __restrict__ n_own) {
  if (st->err_capacity || st->err_range) return;
  const int n_start = st->n_start;
  const int lane = threadIdx.x & 31;
  for (int j = blockIdx.x * 8 + (threadIdx.x >> 5); j < n_start; j += gridDim.x * 8) {
    const int4 pr = __ldg(&perm[j]);
    const int t = slot_trk[pr.x];
    if (t < 0) continue;
    const int s = pr.y >> 16;
    const int nh = n_hits[t];
    const long long h0 = st->hit_off[s] + hit_offset[t + s];
    const uint32_t key = sel_key(nh, t - st->trk_off[s]);
    const uint32_t* ok = own_key + sec[s].off;
    int cnt = 0;
    for (int k = lane; k < nh; k += 32) cnt += (ok[__ldcs(&hit_idx[h0 + k])] == key) ? 1 : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_down_sync(0xffffffffu, cnt, o);
    if (lane == 0) n_own[t] = cnt;
  }
}

// selection rule (integers): shared * 1000 <= max_shared_permille * n_hits
__device__ __forceinline__ bool sel_keep(int nh, int own, int permille) {
  return (long long)(nh - own) * 1000ll <= (long long)permille * (long long)nh;
}

// ---- K6c: per-tile (1024 tracks) sums of (selected, hits of selected) --------------------------------
__global__ void __launch_bounds__(1024)
k_sel_tile_sums(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, const int32_t* __restrict__ n_hits,
                const int32_t* __restrict__ n_own, int2* __restrict__ tile_cnt) {
  __shared__ int ws[33];
  const int n_trk = st->trk_off[T->n_sectors];
  const int t = blockIdx.x * 1024 + threadIdx.x;
  const int nh = t < n_trk ? n_hits[t] : 0;
  const bool keep = t < n_trk && sel_keep(nh, n_own[t], T->sel_permille);
  int ta, tb;
  block_exclusive_scan<int>(keep ? 1 : 0, ws, ta);
  block_exclusive_scan<int>(keep ? nh : 0, ws, tb);
  if (threadIdx.x == 0) tile_cnt[blockIdx.x] = make_int2(ta, tb);
}

// ---- K6d: sector bases of the selected table and of its hit CSR --------------------------------------
__global__ void k_sel_sector_bases(const DevTables* __restrict__ T, DevStatus* __restrict__ st, const int32_t* __restrict__ n_hits,
                                   const int32_t* __restrict__ n_own, const longlong2* __restrict__ tile_off,
                                   const int64_t* __restrict__ tot) {
  const int ns = T->n_sectors;
  const int s = threadIdx.x;
  if (s > ns) return;
  const int n_trk = st->trk_off[ns];
  const int t0 = st->trk_off[s];
  if (t0 >= n_trk) { st->sel_off[s] = (int32_t)tot[0]; st->sel_hit_off[s] = tot[1]; return; }
  const int tile = t0 >> 10;
  long long a = tile_off[tile].x, b = tile_off[tile].y;
  const int permille = T->sel_permille;
  for (int q = tile << 10; q < t0; ++q) {
    const int nh = n_hits[q];
    if (sel_keep(nh, n_own[q], permille)) { a += 1; b += nh; }
  }
  st->sel_off[s] = (int32_t)a;
  st->sel_hit_off[s] = b;
}

// ---- K6e: gather the selected tracks (ascending track number) into the compact table + hit CSR ----------
struct SelOut {
  int32_t* sel_track;        // [n_selected] sector-local track numbers
  TrackOut o;                // compact table: same planes as the S5 table, plane stride = cap
};

__global__ void __launch_bounds__(1024)
k_sel_gather(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, int32_t cap, const int32_t* __restrict__ n_own,
             const longlong2* __restrict__ tile_off, TrackOut in, SelOut out) {
  __shared__ int ws[33];
  const int ns = T->n_sectors;
  const int n_trk = st->trk_off[ns];
  const int t = blockIdx.x * 1024 + threadIdx.x;
  const bool valid = t < n_trk;
  const int nh = valid ? in.n_hits[t] : 0;
  const bool keep = valid && sel_keep(nh, n_own[t], T->sel_permille);
  int ta, tb;
  const int ea = block_exclusive_scan<int>(keep ? 1 : 0, ws, ta);
  const int eb = block_exclusive_scan<int>(keep ? nh : 0, ws, tb);
  const long long k = tile_off[blockIdx.x].x + ea;       // global index in the selected table
  const long long h = tile_off[blockIdx.x].y + eb;       // global index in the selected hit CSR
  long long src_h = 0;
  if (valid) {
    const int s = sector_of_track(st, ns, t);
    const long long hloc = h - st->sel_hit_off[s];
    src_h = st->hit_off[s] + in.hit_offset[t + s];
    if (keep) {
      const size_t cs = (size_t)cap;
      out.sel_track[k] = t - st->trk_off[s];
      out.o.hit_offset[k + s] = (int32_t)hloc;
      out.o.x_ref[k] = in.x_ref[t]; out.o.z_ref[k] = in.z_ref[t]; out.o.chi2[k] = in.chi2[t];
#pragma unroll
      for (int i = 0; i < 5; ++i) out.o.par[i * cs + k] = in.par[i * cs + t];
#pragma unroll
      for (int i = 0; i < 15; ++i) out.o.cov[i * cs + k] = in.cov[i * cs + t];
      out.o.n_hits[k] = nh; out.o.n_fit[k] = in.n_fit[t]; out.o.first_row[k] = in.first_row[t];
      out.o.last_row[k] = in.last_row[t]; out.o.start_hit[k] = in.start_hit[t];
    }
    // closing entry of the sector's hit_offset: written by the sector's last track
    if (t + 1 == st->trk_off[s + 1]) out.o.hit_offset[k + (keep ? 1 : 0) + s] = (int32_t)(hloc + (keep ? nh : 0));
  }
  // hit lists: the warp copies the list of each of its selected tracks together
  const int lane = threadIdx.x & 31;
  unsigned todo = __ballot_sync(0xffffffffu, keep);
  while (todo) {
    const int src = __ffs(todo) - 1;
    todo &= todo - 1;
    const int n = __shfl_sync(0xffffffffu, nh, src);
    const long long from = __shfl_sync(0xffffffffu, src_h, src), to = __shfl_sync(0xffffffffu, h, src);
    for (int q = lane; q < n; q += 32) out.o.hit_idx[to + q] = in.hit_idx[from + q];
  }
}

// sectors without tracks still own a one-entry hit_offset = {0} in the selected table
__global__ void k_sel_close_empty(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, SelOut out) {
  const int s = threadIdx.x;
  if (s >= T->n_sectors) return;
  if (st->trk_off[s] == st->trk_off[s + 1]) out.o.hit_offset[st->sel_off[s] + s] = 0;
}

// ---- K6f: in place: owner[c] = track number decoded from the key (-1: the cluster is in no track) --------
__global__ void __launch_bounds__(256)
k_sel_owner(uint32_t* __restrict__ key_owner, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const uint32_t k = key_owner[i];
    key_owner[i] = k ? (uint32_t)(((1 << kSelTrackBits) - 1) - (int)(k & ((1u << kSelTrackBits) - 1u))) : 0xFFFFFFFFu;
  }
}

// ---- S7: track-residual front end --------------------------------------
// Per cluster: res_trk = the SELECTED track owning it (-1: none), residuals to that track's helix, quantised.
static_assert(sizeof(tpcca_residual) == 16, "tpcca_residual is one 16-byte record");

__global__ void __launch_bounds__(256)
k_res_init(tpcca_residual* __restrict__ o, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    reinterpret_cast<int4*>(o)[i] = make_int4(-1, 0, 0, 0);
}

__device__ __forceinline__ int16_t res_quantise(float r, float inv_q) {
  float v = rintf(__fmul_rn(r, inv_q));       // round half to even
  v = v > 32767.0f ? 32767.0f : v;
  v = v < -32767.0f ? -32767.0f : v;
  return (int16_t)(int)v;
}

// One thread per selected track: the fitted state is transported hit to hit (mean only, the operations of
// kf_prop_mean = DESIGN.md 3.5 Propagate) and every hit the track owns gets its residual.
__global__ void __launch_bounds__(128)
k_residuals(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, const DevStatus* __restrict__ st,
            const float2* __restrict__ syz, const int32_t* __restrict__ row_start, const int32_t* __restrict__ owner,
            SelOut sel, int32_t cap, tpcca_residual* __restrict__ o, float* __restrict__ out_x /*[cap]*/, float* __restrict__ out_p /*[5][cap]*/,
            int32_t* __restrict__ out_ok /*[cap]: S8 needs the state on the last row*/) {
  const int ns = T->n_sectors, n_rows = T->n_rows;
  const int n_sel = st->sel_off[ns];
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n_sel) return;
  int s = 0;
  {
    int lo = 0, hi = ns - 1;
    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (st->sel_off[mid] <= k) lo = mid; else hi = mid - 1; }
    s = lo;
  }
  const int t_local = sel.sel_track[k];
  const size_t cs = (size_t)cap;
  KF f;
  f.x = sel.o.x_ref[k];
  const float z_ref = sel.o.z_ref[k];
  f.p0 = sel.o.par[k]; f.p1 = sel.o.par[cs + k]; f.p2 = sel.o.par[2 * cs + k]; f.p3 = sel.o.par[3 * cs + k]; f.p4 = sel.o.par[4 * cs + k];
  KFConst K;
  K.Bc = T->Bc; K.err2_y = 0.f; K.err2_z = 0.f; K.max_sinphi = T->max_sinphi;
  K.c24 = (float)(1.0 / 24.0); K.c640 = (float)(3.0 / 640.0); K.c12 = (float)(1.0 / 12.0);
  K.ic0 = K.ic1 = K.ic2 = K.ic3 = K.ic4 = 0.f;
  const float inv_q = T->res_inv_q;
  const int nh = sel.o.n_hits[k];
  const int32_t* hl = sel.o.hit_idx + (st->sel_hit_off[s] + sel.o.hit_offset[k + s]);
  const int off = sec[s].off;
  const int32_t* rs = row_start + (size_t)s * (n_rows + 1);
  int r = sel.o.first_row[k];
  bool walked = true;
  // the hit, its cluster and its owner are read one step ahead of the transport (their latency is off the chain)
  int c_n = nh > 0 ? hl[0] : 0;
  float2 h_n = nh > 0 ? __ldg(&syz[off + c_n]) : make_float2(0.f, 0.f);
  int own_n = nh > 0 ? owner[off + c_n] : -1;
  for (int q = 0; q < nh; ++q) {
    const int c = c_n;
    const float2 h = h_n;
    const int own = own_n;
    if (q + 1 < nh) { c_n = hl[q + 1]; h_n = __ldg(&syz[off + c_n]); own_n = owner[off + c_n]; }
    while (r + 1 < n_rows && c >= __ldg(&rs[r + 1])) ++r;     // hits ascend in row
    KFJac J;
    if (!kf_prop_mean(f, __ldg(&T->row_x[r]), K, J)) { walked = false; break; }
    if (own != t_local) continue;
    const float ry = h.x - f.p0;
    const float rz = (h.y - z_ref) - f.p1;
    const int qq = (int)(uint16_t)res_quantise(ry, inv_q) | ((int)(uint16_t)res_quantise(rz, inv_q) << 16);
    reinterpret_cast<int4*>(o)[off + c] = make_int4(t_local, __float_as_int(ry), __float_as_int(rz), qq);   // one 16-byte store
  }
  out_ok[k] = (walked && nh > 0) ? 1 : 0;
  out_x[k] = f.x;
  out_p[k] = f.p0; out_p[cs + k] = f.p1; out_p[2 * cs + k] = f.p2; out_p[3 * cs + k] = f.p3; out_p[4 * cs + k] = f.p4;
}

}  // namespace tpcca
