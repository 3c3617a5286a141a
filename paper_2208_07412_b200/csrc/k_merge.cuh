// S8 cross-sector merging + chain refit.  Works on the compact table
// of the SELECTED tracks (S6) and their outer states (S7 walk).  "k" = global selected index (sector s owns
// [sel_off[s], sel_off[s+1])).
#pragma once
#include "k_select.cuh"

namespace tpcca {

struct MgParams {
  int32_t per_side, max_row_gap, n_zb;      // sectors per side; row gap; z buckets per row of the candidate index
  float ca, sa;                             // cos / sin of the angle between neighbouring sectors
  float dy, dz, ds, zpre;                   // match windows, z pre-cut
  float zb_lo, zb_inv;                      // candidate index: z bucket = clamp(floor((z - zb_lo) * zb_inv), 0, n_zb - 1)
};

struct MgBuf {
  // S7 by-product: state of every selected track on its last row
  float* out_x;           // [CS]
  float* out_p;           // [5][CS]
  int32_t* out_ok;        // [CS]
  // candidate index: selected tracks of a sector bucketed by (first_row, z bucket of z_ref + p1)
  uint32_t* bk_cnt;       // [ns * n_rows * n_zb + 1] counts, then exclusive starts
  int32_t* bk_list;       // [CS] global selected indices, bucket by bucket
  unsigned long long* next_key;   // [CS] best upper partner: score bits << 32 | sector << 23 | track
  unsigned long long* prev_key;   // [CS] best lower partner (atomicMin)
  // outputs, per selected track
  int32_t *next_sec, *next_trk, *prev_sec, *prev_trk;   // [CS]
  int32_t *n_seg, *n_hits, *n_fit, *first_row, *last_row, *frame_seg;   // [CS] merged chain headed here (n_seg = 0: none)
  float *x_ref, *z_ref, *chi2, *par /*[5][CS]*/, *cov /*[15][CS]*/;
};

__device__ __forceinline__ int sector_of_sel(const DevStatus* __restrict__ st, int ns, int k) {
  int lo = 0, hi = ns - 1;
  while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (st->sel_off[mid] <= k) lo = mid; else hi = mid - 1; }
  return lo;
}

__device__ __forceinline__ int mg_zbucket(float z, const MgParams& M) {
  const int b = __float2int_rd(__fmul_rn(__fsub_rn(z, M.zb_lo), M.zb_inv));
  return min(max(b, 0), M.n_zb - 1);
}

// DESIGN.md 3.7 "Rotate" (mean + covariance), every operation in the defined order.
__device__ __forceinline__ bool kf_rotate(KF& s, float ca, float sa, float Bc, float max_sinphi) {
  const float sf = s.p2;
  if (!(fabsf(sf) <= max_sinphi)) return false;
  const float cf = sqrtf(1.0f - sf * sf);
  const float sf2 = sf * ca - cf * sa;
  if (!(fabsf(sf2) <= max_sinphi)) return false;
  const float cf2 = sqrtf(1.0f - sf2 * sf2);
  const float x2 = s.x * ca + s.p0 * sa;
  const float y2 = s.p0 * ca - s.x * sa;
  const float j00 = cf / cf2;
  const float j10 = -((s.p3 * sa) / cf2);
  const float j20 = -((s.p4 * Bc) * sa);
  const float j22 = cf2 / cf;
  const float A00 = j00 * s.c00;
  const float A10 = j10 * s.c00 + s.c10, A11 = j10 * s.c10 + s.c11;
  const float A20 = j20 * s.c00 + j22 * s.c20, A21 = j20 * s.c10 + j22 * s.c21, A22 = j20 * s.c20 + j22 * s.c22;
  const float A30 = s.c30, A31 = s.c31, A32 = s.c32;
  const float A40 = s.c40, A41 = s.c41, A42 = s.c42;
  s.c00 = A00 * j00;
  s.c10 = A10 * j00; s.c11 = A10 * j10 + A11;
  s.c20 = A20 * j00; s.c21 = A20 * j10 + A21; s.c22 = A20 * j20 + A22 * j22;
  s.c30 = A30 * j00; s.c31 = A30 * j10 + A31; s.c32 = A30 * j20 + A32 * j22;
  s.c40 = A40 * j00; s.c41 = A40 * j10 + A41; s.c42 = A40 * j20 + A42 * j22;
  s.x = x2; s.p0 = y2; s.p2 = sf2;
  return true;
}

// ---- K8a: candidate index, pass 1: bucket counts ----------------------------------------------------------
__global__ void __launch_bounds__(256)
k_mg_count(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, SelOut sel, int32_t cap, MgParams M, MgBuf B) {
  const int ns = T->n_sectors, nr = T->n_rows;
  const int n_sel = st->sel_off[ns];
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n_sel) return;
  const int s = sector_of_sel(st, ns, k);
  const float z = sel.o.z_ref[k] + sel.o.par[(size_t)cap + k];
  const int key = (s * nr + sel.o.first_row[k]) * M.n_zb + mg_zbucket(z, M);
  atomicAdd(&B.bk_cnt[key], 1u);
  B.next_key[k] = ~0ull; B.prev_key[k] = ~0ull;
  B.next_sec[k] = -1; B.next_trk[k] = -1; B.prev_sec[k] = -1; B.prev_trk[k] = -1; B.n_seg[k] = 0;
}

// exclusive scan of the bucket counters in place, one block per sector: the first bucket of sector s starts at
// sel_off[s] (every selected track of the sector sits in one of its buckets), so the sectors need no carry
__global__ void __launch_bounds__(1024)
k_mg_scan(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, uint32_t* __restrict__ cnt, int per_sector) {
  __shared__ uint32_t ws[33];
  const int s = blockIdx.x;
  uint32_t* c = cnt + (size_t)s * per_sector;
  uint32_t carry = (uint32_t)st->sel_off[s];
  for (int b0 = 0; b0 < per_sector; b0 += 8192) {
    const int i0 = b0 + threadIdx.x * 8;
    uint32_t v[8], sum = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { v[j] = (i0 + j < per_sector) ? c[i0 + j] : 0u; sum += v[j]; }
    uint32_t total;
    uint32_t run = carry + block_exclusive_scan<uint32_t>(sum, ws, total);
#pragma unroll
    for (int j = 0; j < 8; ++j) { if (i0 + j < per_sector) c[i0 + j] = run; run += v[j]; }
    carry += total;
  }
  if (s == T->n_sectors - 1 && threadIdx.x == 0) c[per_sector] = carry;      // closing entry
}

// pass 2: scatter (the order inside a bucket is arbitrary: no result depends on it)
__global__ void __launch_bounds__(256)
k_mg_scatter(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, SelOut sel, int32_t cap, MgParams M, MgBuf B,
             uint32_t* __restrict__ cursor) {
  const int ns = T->n_sectors, nr = T->n_rows;
  const int n_sel = st->sel_off[ns];
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n_sel) return;
  const int s = sector_of_sel(st, ns, k);
  const float z = sel.o.z_ref[k] + sel.o.par[(size_t)cap + k];
  const int key = (s * nr + sel.o.first_row[k]) * M.n_zb + mg_zbucket(z, M);
  B.bk_list[B.bk_cnt[key] + atomicAdd(&cursor[key], 1u)] = k;
}

// ---- K8b: matching.  One thread per selected track a: its best upper partner; atomicMin for the partner's best lower
__global__ void __launch_bounds__(128)
k_mg_match(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, SelOut sel, int32_t cap, MgParams M, MgBuf B) {
  const int ns = T->n_sectors, nr = T->n_rows;
  const int n_sel = st->sel_off[ns];
  const int ka = blockIdx.x * blockDim.x + threadIdx.x;
  if (ka >= n_sel || !B.out_ok[ka]) return;
  const int per = M.per_side;
  if (per < 2 || ns % per != 0) return;
  const size_t cs = (size_t)cap;
  const int s = sector_of_sel(st, ns, ka);
  const int ia = ka - st->sel_off[s];
  const int side = s / per, loc = s % per;
  const int last_a = sel.o.last_row[ka];
  const float zref_a = sel.o.z_ref[ka];
  KFConst K;
  K.Bc = T->Bc; K.err2_y = 0.f; K.err2_z = 0.f; K.max_sinphi = T->max_sinphi;
  K.c24 = (float)(1.0 / 24.0); K.c640 = (float)(3.0 / 640.0); K.c12 = (float)(1.0 / 12.0);
  K.ic0 = K.ic1 = K.ic2 = K.ic3 = K.ic4 = 0.f;
  KF out;
  out.x = B.out_x[ka];
  out.p0 = B.out_p[ka]; out.p1 = B.out_p[cs + ka]; out.p2 = B.out_p[2 * cs + ka]; out.p3 = B.out_p[3 * cs + ka]; out.p4 = B.out_p[4 * cs + ka];
  kf_reset_cov(out, K);                     // zero covariance: only the mean is used
  const float za = zref_a + out.p1;
  // One bucket more on each side than fl(za -+ zpre) fall in: the pre-cut below is |fl(zb - za)| <= zpre, and a zb one
  // ulp beyond fl(za + zpre) can still pass it after rounding while sitting across a bucket edge.  The extra
  // buckets only add candidates that the exact pre-cut then rejects, so no other result changes.
  const int zb0 = max(mg_zbucket(za - M.zpre, M) - 1, 0), zb1 = min(mg_zbucket(za + M.zpre, M) + 1, M.n_zb - 1);
  unsigned long long best = ~0ull;
  for (int dir = 0; dir < 2; ++dir) {
    const int nsec = side * per + (dir == 0 ? (loc + 1) % per : (loc + per - 1) % per);
    if (nsec == s || (per == 2 && dir == 1)) continue;
    KF rot = out;
    if (!kf_rotate(rot, M.ca, dir == 0 ? M.sa : -M.sa, K.Bc, K.max_sinphi)) continue;
    const int k0 = st->sel_off[nsec];
    for (int row = last_a + 1; row <= min(last_a + M.max_row_gap, nr - 1); ++row) {
      const uint32_t* bc = B.bk_cnt + (size_t)(nsec * nr + row) * M.n_zb;
      const uint32_t e = bc[zb1 + 1];
      for (uint32_t q = bc[zb0]; q < e; ++q) {
        const int kb = B.bk_list[q];
        const float zref_b = sel.o.z_ref[kb], p1b = sel.o.par[cs + kb];
        const float zb = zref_b + p1b;
        if (!(fabsf(zb - za) <= M.zpre)) continue;
        KF t = rot;
        KFJac J;
        if (!kf_prop_mean(t, sel.o.x_ref[kb], K, J)) continue;
        const float dy = sel.o.par[kb] - t.p0;
        const float dz = (zref_b - zref_a) + (p1b - t.p1);
        const float ds = sel.o.par[2 * cs + kb] - t.p2;
        if (!(fabsf(dy) <= M.dy && fabsf(dz) <= M.dz && fabsf(ds) <= M.ds)) continue;
        const float qy = dy / M.dy, qz = dz / M.dz, qs = ds / M.ds;
        const float sc = qy * qy + qz * qz + qs * qs;
        const unsigned long long hi = (unsigned long long)__float_as_uint(sc) << 32;
        const unsigned long long kn = hi | ((unsigned long long)nsec << kSelTrackBits) | (unsigned long long)(kb - k0);
        best = kn < best ? kn : best;
        atomicMin(&B.prev_key[kb], hi | ((unsigned long long)s << kSelTrackBits) | (unsigned long long)ia);
      }
    }
  }
  B.next_key[ka] = best;
}

// ---- K8c: a link is kept iff it is mutual ---------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_mg_link(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, MgBuf B) {
  const int ns = T->n_sectors;
  const int n_sel = st->sel_off[ns];
  const int ka = blockIdx.x * blockDim.x + threadIdx.x;
  if (ka >= n_sel) return;
  const unsigned long long kn = B.next_key[ka];
  if (kn == ~0ull) return;
  const int s = sector_of_sel(st, ns, ka);
  const int ia = ka - st->sel_off[s];
  const uint32_t lo = (uint32_t)kn;
  const int nsec = (int)(lo >> kSelTrackBits), ib = (int)(lo & ((1u << kSelTrackBits) - 1u));
  const int kb = st->sel_off[nsec] + ib;
  const uint32_t back = (uint32_t)B.prev_key[kb];
  if ((int)(back >> kSelTrackBits) == s && (int)(back & ((1u << kSelTrackBits) - 1u)) == ia) {
    B.next_sec[ka] = nsec; B.next_trk[ka] = ib;
    B.prev_sec[kb] = s; B.prev_trk[kb] = ia;
  }
}

// ---- K8c': the heads of chains (no partner below, one above), compacted (any order: outputs are indexed by the head)
__global__ void __launch_bounds__(256)
k_mg_heads(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, MgBuf B, int32_t* __restrict__ head_list,
           uint32_t* __restrict__ n_heads) {
  const int n_sel = st->sel_off[T->n_sectors];
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const bool head = k < n_sel && B.prev_sec[k] == -1 && B.next_sec[k] != -1;
  const unsigned m = __ballot_sync(0xffffffffu, head);
  if (!m) return;
  const int lane = threadIdx.x & 31;
  uint32_t base = 0;
  if (lane == 0) base = atomicAdd(n_heads, (uint32_t)__popc(m));
  base = __shfl_sync(0xffffffffu, base, 0);
  if (head) head_list[base + __popc(m & ((1u << lane) - 1u))] = k;
}

// ---- K8d: refit of the chains.  One thread per chain head --------------------------------------------------------
__global__ void __launch_bounds__(128)
k_mg_refit(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, const DevStatus* __restrict__ st,
           const float2* __restrict__ syz, const int32_t* __restrict__ row_start, SelOut sel, int32_t cap, MgParams M, MgBuf B,
           const int32_t* __restrict__ head_list, const uint32_t* __restrict__ n_heads) {
  const int ns = T->n_sectors, nr = T->n_rows;
  const int ih = blockIdx.x * blockDim.x + threadIdx.x;
  if (ih >= (int)*n_heads) return;
  const int kh = head_list[ih];
  const size_t cs = (size_t)cap;
  // walk up to the top segment
  int n_seg = 1, ktop = kh;
  while (B.next_sec[ktop] != -1) { ktop = st->sel_off[B.next_sec[ktop]] + B.next_trk[ktop]; ++n_seg; }
  KFConst K;
  K.Bc = T->Bc; K.err2_y = T->err2_y; K.err2_z = T->err2_z; K.max_sinphi = T->max_sinphi;
  K.c24 = (float)(1.0 / 24.0); K.c640 = (float)(3.0 / 640.0); K.c12 = (float)(1.0 / 12.0);
  K.ic0 = T->init_cov[0]; K.ic1 = T->init_cov[1]; K.ic2 = T->init_cov[2]; K.ic3 = T->init_cov[3]; K.ic4 = T->init_cov[4];
  KF f;
  f.x = B.out_x[ktop];
  f.p0 = B.out_p[ktop]; f.p1 = B.out_p[cs + ktop]; f.p2 = B.out_p[2 * cs + ktop]; f.p3 = B.out_p[3 * cs + ktop]; f.p4 = B.out_p[4 * cs + ktop];
  kf_reset_cov(f, K);
  bool ok = B.out_ok[ktop] != 0;
  KF snap = f;
  bool have_snap = false;
  int n_hits = 0, first = -1, last = -1, g = n_seg - 1, g_snap = n_seg - 1;
  int kcur = ktop, kup = -1;
  while (ok) {
    const int s = sector_of_sel(st, ns, kcur);
    const float zref = sel.o.z_ref[kcur];
    if (kup >= 0) {
      const int up = sector_of_sel(st, ns, kup);
      const bool up_is_next = (up % M.per_side) == ((s % M.per_side) + 1) % M.per_side;
      if (!kf_rotate(f, M.ca, up_is_next ? -M.sa : M.sa, K.Bc, K.max_sinphi)) break;
      f.p1 = f.p1 + (sel.o.z_ref[kup] - zref);
    }
    const int nh = sel.o.n_hits[kcur];
    const int32_t* hl = sel.o.hit_idx + (st->sel_hit_off[s] + sel.o.hit_offset[kcur + s]);
    const int off = sec[s].off;
    const int32_t* rs = row_start + (size_t)s * (nr + 1);
    int r = sel.o.last_row[kcur];
    for (int q = nh - 1; q >= 0; --q) {
      const int c = hl[q];
      while (r > 0 && c < __ldg(&rs[r])) --r;            // hits descend in row
      const float2 h = __ldg(&syz[off + c]);
      if (!kf_propagate(f, __ldg(&T->row_x[r]), K)) { ok = false; break; }
      kf_update(f, h.x, h.y - zref, K);
      snap = f; have_snap = true; g_snap = g;
      if (last < 0) last = r;
      first = r;
      ++n_hits;
    }
    if (!ok || B.prev_sec[kcur] == -1) break;
    kup = kcur;
    kcur = st->sel_off[B.prev_sec[kcur]] + B.prev_trk[kcur];
    --g;
  }
  if (!have_snap) return;
  // z_ref of the segment the refit ended in: walk g_snap links up from the head
  int kz = kh;
  for (int i = 0; i < g_snap; ++i) kz = st->sel_off[B.next_sec[kz]] + B.next_trk[kz];
  B.n_seg[kh] = n_seg; B.n_hits[kh] = n_hits; B.n_fit[kh] = snap.n; B.first_row[kh] = first; B.last_row[kh] = last;
  B.frame_seg[kh] = g_snap;
  B.x_ref[kh] = snap.x; B.z_ref[kh] = sel.o.z_ref[kz]; B.chi2[kh] = snap.chi2;
  B.par[kh] = snap.p0; B.par[cs + kh] = snap.p1; B.par[2 * cs + kh] = snap.p2; B.par[3 * cs + kh] = snap.p3; B.par[4 * cs + kh] = snap.p4;
  const float cv[15] = {snap.c00, snap.c10, snap.c11, snap.c20, snap.c21, snap.c22, snap.c30, snap.c31, snap.c32, snap.c33,
                        snap.c40, snap.c41, snap.c42, snap.c43, snap.c44};
#pragma unroll
  for (int i = 0; i < 15; ++i) B.cov[i * cs + kh] = cv[i];
}

}  // namespace tpcca
