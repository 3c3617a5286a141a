// S2 neighbour finder, S3 link cleaner, S4 start hits.
#pragma once
#include "k_grid.cuh"

namespace tpcca {

__device__ __forceinline__ int row_search(const int32_t* __restrict__ rs, int n_rows, int p) {
  int lo = 0, hi = n_rows - 1;               // largest r with rs[r] <= p
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (__ldg(&rs[mid]) <= p) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// ---- S2 tiling and staging -------------------------------------------------------
// A tile = kNfTile consecutive sorted clusters of ONE (sector, row).  Because the sort key is
// (row, bz, by, id), the window candidates of a whole tile in row r+1 (r-1) are ONE contiguous run
// of sorted clusters (the z slices S_lo..S_hi of that row) and their bin_start entries are one
// contiguous run as well.  k_nf_plan writes one descriptor per tile; k_neighbours stages the two
// cluster runs and the two bin_start runs of the next tile in shared memory with 1-D bulk async
// copies (TMA, mbarrier completion) while the current tile is searched entirely in shared memory.
#ifndef TPCCA_NF_T2
#define TPCCA_NF_T2 2      // window-test candidates per loop trip
#endif
#ifndef TPCCA_NF_K
#define TPCCA_NF_K 10
#endif
#ifndef TPCCA_NF_ARENA
#define TPCCA_NF_ARENA 8448
#endif
constexpr int kNfK = TPCCA_NF_K;          // window hits cached per side and thread in shared memory (<= 15): normal occupancy
constexpr int kNfKDense = 15;             // ... of the kernel instance used for dense time frames (tpcca_create chooses)
static_assert(TPCCA_NF_K <= 15 && TPCCA_NF_TILE <= 256, "work-item encoding: 8 bits cluster, 4 bits hit row, 4 bits nd");
constexpr int kNfThreads = kNfTile;       // one thread per cluster of the tile
constexpr int kNfArena = TPCCA_NF_ARENA;  // bytes of one staging buffer: [up clusters | down clusters | up bins | down bins]
constexpr int kNfMaxCn = 1022;            // staged clusters per side (staged indices are packed in 10 bits)
constexpr int kNfMaxRun = 63;             // window candidates per side handled by the packed fast path

enum { NF_STAGED = 0, NF_NOLINK = 1, NF_GLOBAL = 2, NF_STAGED_C = 3 };   // STAGED_C: clusters staged, bins read from global memory

struct NfSide {        // staging of one neighbour row for one tile
  int32_t c0;          // sector-local sorted position of staged cluster 0 ((sec_off + c0) is even; may be -1)
  int32_t cn;          // staged clusters (even)
  uint32_t b0;         // global bin_start index of staged entry 0 (multiple of 4)
  int32_t bn;          // staged entries (multiple of 4)
  int32_t s0;          // first staged z slice
  int32_t ds_shift;    // (last staged slice - s0) | (index of slice s0's first entry in the staged run) << 24
};
struct NfTileDesc {    // 64 bytes
  int32_t p0;          // global index (concatenated arrays) of the tile's first cluster
  int32_t n;           // clusters in the tile (1..kNfTile)
  int32_t rsf;         // row | sector << 8 | flag << 16
  int32_t sec_off;     // global index of the sector's sorted position 0
  NfSide up, dn;
};
static_assert(sizeof(NfTileDesc) == 64, "NfTileDesc must be 64 bytes");

struct NfTable { NfConst row[kMaxRows]; };   // by-value kernel parameter (constant bank): 28 KB

// ---- mbarrier / bulk-copy primitives (PTX; sm_90+ syntax, SASS: SYNCS / UBLKCP) ------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}

// ---- K2a: tile planner, one block per (sector, row), one thread per tile of that row ------------
// Staged slices of the neighbour row rn for a tile whose clusters have own-row slices b_first..b_last:
// S_lo = slice of (lower z edge of b_first) - (hz + margin) - slack, S_hi likewise.  The bound is a
// performance device only: k_neighbours re-checks every cluster's exact slice range against
// [S_lo, S_hi] and sends the cluster to the global-memory path if it is not covered.
__device__ __forceinline__ void nf_plan_side(NfSide& o, int& flag, const DevTables* __restrict__ T, int rn, float hm,
                                             int b_first, int b_last, int nz_r, float bin_r, uint32_t bs_off,
                                             int sec_off, const uint32_t* __restrict__ bin_start) {
  const float zlo = T->grid_z_lo, ibz = T->inv_bz[rn];
  const int nzh = T->nz[rn] - 1, ny = T->ny[rn];
  int s_lo = 0, s_hi = nzh;
  if (b_first > 0) {
    const float ze = (float)b_first * bin_r + zlo;
    s_lo = bin_range(ze - hm - (0.02f + 1e-6f * fabsf(ze)), zlo, ibz, nzh);
  }
  if (b_last < nz_r - 1) {
    const float ze = (float)(b_last + 1) * bin_r + zlo;
    s_hi = bin_range(ze + hm + (0.02f + 1e-6f * fabsf(ze)), zlo, ibz, nzh);
  }
  const uint32_t gb_lo = bs_off + (uint32_t)(T->bin_base[rn] + s_lo * ny);
  const uint32_t gb_hi = bs_off + (uint32_t)(T->bin_base[rn] + (s_hi + 1) * ny);   // inclusive: end of slice s_hi
  const uint32_t b0 = gb_lo & ~3u;
  const int bn = (int)((gb_hi + 1u - b0 + 3u) & ~3u);
  const int c_lo = (int)bin_start[gb_lo], c_hi = (int)bin_start[gb_hi];
  const int c0 = c_lo - ((sec_off + c_lo) & 1);
  const int cn = (c_hi - c0 + 1) & ~1;
  o.c0 = c0; o.cn = cn; o.b0 = b0; o.bn = bn; o.s0 = s_lo;
  o.ds_shift = (s_hi - s_lo) | ((int)(gb_lo - b0) << 24);
  if (cn > kNfMaxCn || (s_hi - s_lo) >= (1 << 24)) flag = NF_GLOBAL;
}

__global__ void __launch_bounds__(128)
k_nf_plan(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, const float2* __restrict__ syz,
          const uint32_t* __restrict__ bin_start, const int32_t* __restrict__ row_start,
          const int32_t* __restrict__ nf_tile_start, NfTileDesc* __restrict__ desc) {
  const int n_rows = T->n_rows;
  const int n_sr = T->n_sectors * n_rows;
  const uint32_t nbp1 = (uint32_t)T->bins_per_sector + 1u;
  for (int i = blockIdx.x; i < n_sr; i += gridDim.x) {
    const int t0 = nf_tile_start[i], t1 = nf_tile_start[i + 1];
    if (t1 == t0) continue;
    const int s = i / n_rows, r = i - s * n_rows;
    const int rs0 = row_start[s * (n_rows + 1) + r], rs1 = row_start[s * (n_rows + 1) + r + 1];
    const int sec_off = sec[s].off;
    const uint32_t bs_off = (uint32_t)s * nbp1;
    const bool edge = (r < 1 || r > n_rows - 2);
    const float zlo = T->grid_z_lo, ibz = T->inv_bz[r];
    const float bin_r = 1.0f / ibz;
    const int nz_r = T->nz[r];
    for (int t = t0 + threadIdx.x; t < t1; t += blockDim.x) {
      NfTileDesc d;
      const int pl0 = rs0 + (t - t0) * kNfTile;
      d.p0 = sec_off + pl0;
      d.n = min(kNfTile, rs1 - pl0);
      d.sec_off = sec_off;
      int flag = edge ? NF_NOLINK : NF_STAGED;
      d.up = NfSide{0, 0, 0u, 0, 0, 0};
      d.dn = d.up;
      if (!edge) {
        const int b_first = bin_range(syz[d.p0].y, zlo, ibz, nz_r - 1);
        const int b_last = bin_range(syz[d.p0 + d.n - 1].y, zlo, ibz, nz_r - 1);
        nf_plan_side(d.up, flag, T, r + 1, T->hz_up[r] + T->margin, b_first, b_last, nz_r, bin_r, bs_off, sec_off, bin_start);
        nf_plan_side(d.dn, flag, T, r - 1, T->hz_dn[r] + T->margin, b_first, b_last, nz_r, bin_r, bs_off, sec_off, bin_start);
        if (flag == NF_STAGED && 8 * (d.up.cn + d.dn.cn) + 4 * (d.up.bn + d.dn.bn) > kNfArena)
          flag = (8 * (d.up.cn + d.dn.cn) <= kNfArena) ? NF_STAGED_C : NF_GLOBAL;
      }
      d.rsf = r | (s << 8) | (flag << 16);
      desc[t] = d;
    }
  }
}

// ---- exact slow path (global memory) ---------------------------------------------------------------
// visit every window candidate of one side (A, B, C = the side's NfConst groups): plain nested loops
template <class F>
__device__ __forceinline__ void nf_for_each(const float2 c, const float4 A, const float4 B, const int4 C,
                                            const uint32_t* __restrict__ bs, const float2* __restrict__ yz, F fn) {
  const int by0 = bin_range(__fsub_rn(c.x, A.z), B.x, B.y, C.x), by1 = bin_range(__fadd_rn(c.x, A.z), B.x, B.y, C.x);
  const int bz0 = bin_range(__fsub_rn(c.y, A.w), B.w, B.z, C.y), bz1 = bin_range(__fadd_rn(c.y, A.w), B.w, B.z, C.y);
  for (int bz = bz0; bz <= bz1; ++bz) {
    const uint32_t* bp = bs + C.w + bz * C.z;
    const uint32_t e = __ldg(&bp[by1 + 1]);
    for (uint32_t q = __ldg(&bp[by0]); q < e; ++q) {
      const float2 v = __ldg(&yz[q]);
      const float dy = __fsub_rn(v.x, c.x), dz = __fsub_rn(v.y, c.y);
      if (fabsf(dy) <= A.x && fabsf(dz) <= A.y) fn(q, dy, dz);
    }
  }
}

// Slow path of S2 (global memory, exact in every case: any number of candidates, ties by original
// id): the full U x D product by nested rescans of both windows.  Taken by clusters whose windows
// are not covered by the staged runs, hold more than kNfK hits or kNfMaxRun candidates on a side,
// or whose best score is tied.
__device__ __noinline__ void nf_slow(const float2 c, const NfConst& kc, const uint32_t* __restrict__ bs,
                                     const float2* __restrict__ yz, const int32_t* __restrict__ ord,
                                     float& best, int32_t& bu, int32_t& bd) {
  const float4 dA = kc.dA, dB = kc.dB, uA = kc.uA, uB = kc.uB, g = kc.g;
  const int4 dC = kc.dC, uC = kc.uC;
  bu = -1; bd = -1; best = 0.0f;
  nf_for_each(c, uA, uB, uC, bs, yz, [&](uint32_t u, float dyu, float dzu) {
    const float Ay = __fmul_rn(dyu, g.y), Az = __fmul_rn(dzu, g.y);
    nf_for_each(c, dA, dB, dC, bs, yz, [&](uint32_t d, float dyd, float dzd) {
      const float ay = __fsub_rn(Ay, __fmul_rn(-dyd, g.x));
      const float az = __fsub_rn(Az, __fmul_rn(-dzd, g.x));
      const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
      bool better;
      if (bu < 0) better = true;
      else if (sc < best) better = true;
      else if (sc == best) {
        const int32_t ou = __ldg(&ord[u]), obu = __ldg(&ord[bu]);
        better = (ou != obu) ? (ou < obu) : (__ldg(&ord[d]) < __ldg(&ord[bd]));
      } else better = false;
      if (better) { best = sc; bu = (int32_t)u; bd = (int32_t)d; }
    });
  });
}

// ---- fast path, phase 0: the candidate runs of one side as a packed descriptor ----------------------
// A window touches nsl = 2 (3 when it straddles a bin edge by less than the margin) z slices of the
// neighbour row; in each slice its y range of bins is ONE run of sorted clusters.  The runs are
// addressed by a flat candidate index j in [0, tot): staged index = q + j + (j >= n0 ? o1 : 0) +
// (j >= n01 ? o2 : 0).  w0 = q | n0 << 10 | o1 << 16 | n01 << 26,  w1 = o2 | tot << 10.
// Returns false if the window is not covered by the staged slices, spans more than 3 slices or holds
// more than kNfMaxRun candidates.
__device__ __forceinline__ bool nf_runs(const float2 c, const float4 A, const float4 B, const int4 C, const NfSide& sd,
                                        const uint32_t* __restrict__ sB, uint32_t& w0, uint32_t& w1, int& tot) {
  const int by0 = bin_range(__fsub_rn(c.x, A.z), B.x, B.y, C.x), by1 = bin_range(__fadd_rn(c.x, A.z), B.x, B.y, C.x);
  const int bz0 = bin_range(__fsub_rn(c.y, A.w), B.w, B.z, C.y), bz1 = bin_range(__fadd_rn(c.y, A.w), B.w, B.z, C.y);
  const int ds = sd.ds_shift & 0xffffff, shift = sd.ds_shift >> 24;
  const int k0 = bz0 - sd.s0, nsl = bz1 - bz0;          // nsl = slices - 1
  w0 = 0; w1 = 0; tot = 0;
  if (k0 < 0 || bz1 - sd.s0 > ds || nsl > 2) return false;
  const uint32_t* bp = sB + shift + k0 * C.z + by0;
  const int w = by1 + 1 - by0;
  const int qa = (int)bp[0], ea = (int)bp[w];
  int qb = ea, eb = ea, qc, ec;
  if (nsl >= 1) { qb = (int)bp[C.z]; eb = (int)bp[C.z + w]; }
  qc = eb; ec = eb;
  if (nsl >= 2) { qc = (int)bp[2 * C.z]; ec = (int)bp[2 * C.z + w]; }
  const int n0 = ea - qa, n01 = n0 + (eb - qb);
  tot = n01 + (ec - qc);
  if (tot > kNfMaxRun) return false;
  w0 = (uint32_t)(qa - sd.c0) | (uint32_t)n0 << 10 | (uint32_t)(qb - ea) << 16 | (uint32_t)n01 << 26;
  w1 = (uint32_t)(qc - eb) | (uint32_t)tot << 10;
  return true;
}

// ---- shared-memory accessors on 32-bit shared addresses (no 64-bit pointer arithmetic in the loops) --
__device__ __forceinline__ float2 lds_f2(uint32_t a) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts_f2(uint32_t a, float x, float y) {
  asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(x), "f"(y) : "memory");
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t a) {
  uint16_t v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts_u16(uint32_t a, uint32_t v) {
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((uint16_t)v) : "memory");
}

constexpr uint32_t kVecRow = 8u * kNfThreads;   // bytes between consecutive rows of the hit-vector cache
constexpr uint32_t kIdxRow = 2u * kNfThreads;   // ... of the hit-index cache

// ---- fast path, phase A: window test of the tot candidates of one side ------------------------------
// sC = shared address of the side's staged cluster run, (hy, hz) the exact window, scale = +dxd (up
// side) or -dxu (down side: (y_c - y_d) * dxu = -((y_d - y_c) * dxu), exact).  Hits go to the thread's
// cache column: vector (dy * scale, dz * scale) at pv + k * kVecRow, staged index at pi + k * kIdxRow.
// Returns the number of hits (may exceed kNfK; only the first kNfK are cached).
template <int K>
__device__ __forceinline__ int nf_test_runs(const float2 c, uint32_t w0, uint32_t w1, uint32_t sC, float hy, float hz,
                                            float scale, uint32_t pv, uint32_t pi) {
  const int n0 = (w0 >> 10) & 63, n01 = w0 >> 26, tot = w1 >> 10;
  const uint32_t o1 = 8u * ((w0 >> 16) & 1023u), o2 = 8u * (w1 & 1023u);
  uint32_t a = sC + 8u * (w0 & 1023u);
  const uint32_t pv_end = pv + K * kVecRow;
  int n = 0;
  // kT candidates per trip: their shared-memory loads are issued before the first test (independent chains)
  constexpr int kT = TPCCA_NF_T2;
#pragma unroll 1
  for (int j = 0; j < tot; j += kT) {
    uint32_t aa[kT];
    float2 v[kT];
#pragma unroll
    for (int k = 0; k < kT; ++k) {
      if (j + k == n0) a += o1;
      if (j + k == n01) a += o2;
      aa[k] = (k == 0 || j + k < tot) ? a : aa[0];
      a += 8u;
    }
#pragma unroll
    for (int k = 0; k < kT; ++k) v[k] = lds_f2(aa[k]);
#pragma unroll
    for (int k = 0; k < kT; ++k) {
      const float dy = __fsub_rn(v[k].x, c.x), dz = __fsub_rn(v[k].y, c.y);
      if ((k == 0 || j + k < tot) && fabsf(dy) <= hy && fabsf(dz) <= hz) {
        if (pv != pv_end) {
          sts_f2(pv, __fmul_rn(dy, scale), __fmul_rn(dz, scale));
          sts_u16(pi, (aa[k] - sC) >> 3);
          pv += kVecRow; pi += kIdxRow;
        }
        ++n;
      }
    }
  }
  return n;
}

// ---- medium path: more than kNfK hits on a side (dense regions) -------------------------------------
// Nested loops over the staged candidate runs of both sides (no hit cache): the U x D product in the
// order and arithmetic of nf_slow, in shared memory.  Returns false on an exact score tie (decided by
// original ids in nf_slow).  iu / id are staged indices.
__device__ __noinline__ bool nf_medium(const float2 c, uint32_t wu0, uint32_t wu1, uint32_t wd0, uint32_t wd1, uint32_t sUC,
                                       uint32_t sDC, const float4 uA, const float4 dA, const float4 g, float& best,
                                       int& iu, int& id) {
  const int un0 = (wu0 >> 10) & 63, un01 = wu0 >> 26, utot = wu1 >> 10;
  const uint32_t uo1 = 8u * ((wu0 >> 16) & 1023u), uo2 = 8u * (wu1 & 1023u);
  const int dn0 = (wd0 >> 10) & 63, dn01 = wd0 >> 26, dtot = wd1 >> 10;
  const uint32_t do1 = 8u * ((wd0 >> 16) & 1023u), do2 = 8u * (wd1 & 1023u);
  bool have = false, tie = false;
  best = 0.0f; iu = -1; id = -1;
  uint32_t au = sUC + 8u * (wu0 & 1023u);
#pragma unroll 1
  for (int ju = 0; ju < utot; ++ju, au += 8u) {
    if (ju == un0) au += uo1;
    if (ju == un01) au += uo2;
    const float2 u = lds_f2(au);
    const float dyu = __fsub_rn(u.x, c.x), dzu = __fsub_rn(u.y, c.y);
    if (!(fabsf(dyu) <= uA.x && fabsf(dzu) <= uA.y)) continue;
    const float Ay = __fmul_rn(dyu, g.y), Az = __fmul_rn(dzu, g.y);
    uint32_t ad = sDC + 8u * (wd0 & 1023u);
#pragma unroll 1
    for (int jd = 0; jd < dtot; ++jd, ad += 8u) {
      if (jd == dn0) ad += do1;
      if (jd == dn01) ad += do2;
      const float2 d = lds_f2(ad);
      const float dyd = __fsub_rn(d.x, c.x), dzd = __fsub_rn(d.y, c.y);
      if (!(fabsf(dyd) <= dA.x && fabsf(dzd) <= dA.y)) continue;
      const float ay = __fsub_rn(Ay, __fmul_rn(-dyd, g.x));
      const float az = __fsub_rn(Az, __fmul_rn(-dzd, g.x));
      const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
      if (have && sc == best) tie = true;
      if (!have || sc < best) { have = true; best = sc; iu = (int)((au - sUC) >> 3); id = (int)((ad - sDC) >> 3); }
    }
  }
  return !tie;
}

template <int K>
struct NfSmem {
  alignas(128) unsigned char arena[kNfArena];   // staging buffer (TMA destination): [up clusters | down clusters | up bins | down bins]
  float2 vec[2 * K][kNfThreads];      // cached hits: rows [0, K) down side, [K, 2K) up side; column = cluster of the tile
  uint16_t hidx[2 * K][kNfThreads];   // staged indices of the cached hits
  uint16_t items[K * kNfThreads];           // pair work items (one per up-side hit): cluster | hit row << 8 | nd << 12
  int hist[2][16], cnt[2][16];           // items per nd (work key) / emission cursors, two consecutive tiles
  NfTileDesc desc[4];
  uint64_t full;
};

// ---- K2b: neighbour finder --------------------------------------------------
// For cluster c of row r (1 <= r <= n_rows-2): over U x D (exact windows in rows r+1, r-1) the
// pair minimising score = ay^2 + az^2, ay = (yu-yc)*dxd - (yc-yd)*dxu; ties -> smallest original
// id of u, then of d; stored if score <= nf_cut[r].
// Persistent blocks walk the tile list with a grid stride (tiles in flight are neighbours in memory,
// so the three-fold reuse of a row stays in L2).  Per tile:
//   phase A  thread t = cluster t: bin ranges of both windows, candidate runs from the staged
//            bin_start entries, window tests of both sides; hits cached in the thread's column.
//   phase B  the nu x nd pair scores are NOT looped per cluster (nu * nd has a long tail: mean 3.7,
//            1 % above 24): every up-side hit becomes a work item (cluster, hit row, nd), the items
//            are counting-sorted by nd in shared memory, and thread i scores item i against the nd
//            down-side hits of its cluster, so the lanes of a warp run the same trip count (<= kNfK).
//   phase C  thread t = cluster t: minimum over its nu item results, cut, coalesced link stores.
// The staged runs of tile i+1 are fetched by bulk async copies (issued by thread 0 right after the
// barrier that ends phase A of tile i, the only phase that reads the staging buffer); per-row
// constants come from the constant bank (NfTable is a by-value kernel parameter).
#ifndef TPCCA_NF_BPS
#define TPCCA_NF_BPS 5
#endif
template <int K>
__global__ void __launch_bounds__(kNfThreads, K == kNfK ? TPCCA_NF_BPS : 4)
k_neighbours(const __grid_constant__ NfTable tab, const float2* __restrict__ syz,
             const uint32_t* __restrict__ bin_start, const int32_t* __restrict__ order, uint32_t nbp1,
             const int32_t* __restrict__ n_tiles_ptr, const NfTileDesc* __restrict__ desc,
             int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  extern __shared__ __align__(128) unsigned char nf_smem_raw[];
  NfSmem<K>& S = *reinterpret_cast<NfSmem<K>*>(nf_smem_raw);
  const int tid = threadIdx.x;
  const int n_tiles = __ldg(n_tiles_ptr);
  const int stride = gridDim.x;
  const int first = blockIdx.x;
  if (first >= n_tiles) return;
  if (tid == 0) { mbar_init(&S.full, 1); fence_mbar_init(); }
  if (tid < 64) (&S.hist[0][0])[tid] = 0;            // hist[2][16] and cnt[2][16] are contiguous
  if (tid < 48) {      // descriptors of the block's first three tiles
    const int k = tid >> 4, t = first + k * stride;
    if (t < n_tiles) reinterpret_cast<int32_t*>(&S.desc[k])[tid & 15] = __ldg(reinterpret_cast<const int32_t*>(&desc[t]) + (tid & 15));
  }
  __syncthreads();
  auto issue = [&](const NfTileDesc& d) {      // thread 0 only
    const int flag = d.rsf >> 16;
    uint32_t bytes = 0;
    if (flag == NF_STAGED) bytes = 8u * (uint32_t)(d.up.cn + d.dn.cn) + 4u * (uint32_t)(d.up.bn + d.dn.bn);
    else if (flag == NF_STAGED_C) bytes = 8u * (uint32_t)(d.up.cn + d.dn.cn);
    mbar_arrive_expect_tx(&S.full, bytes);
    if (bytes) {
      unsigned char* a = S.arena;
      if (d.up.cn) bulk_g2s(a, syz + (d.sec_off + d.up.c0), 8u * d.up.cn, &S.full);
      if (d.dn.cn) bulk_g2s(a + 8 * d.up.cn, syz + (d.sec_off + d.dn.c0), 8u * d.dn.cn, &S.full);
      if (flag == NF_STAGED) {
        unsigned char* b = a + 8 * (d.up.cn + d.dn.cn);
        if (d.up.bn) bulk_g2s(b, bin_start + d.up.b0, 4u * d.up.bn, &S.full);
        if (d.dn.bn) bulk_g2s(b + 4 * d.up.bn, bin_start + d.dn.b0, 4u * d.dn.bn, &S.full);
      }
    }
  };
  if (tid == 0) issue(S.desc[0]);
  float2 c_next = make_float2(0.f, 0.f);
  if (tid < S.desc[0].n) c_next = __ldg(&syz[S.desc[0].p0 + tid]);
  const uint32_t sArena = smem_u32(S.arena);
  const uint32_t sVecD = smem_u32(&S.vec[0][0]), sVecU = smem_u32(&S.vec[K][0]);
  const uint32_t sIdxD = smem_u32(&S.hidx[0][0]), sIdxU = smem_u32(&S.hidx[K][0]);
  int it = 0;
  for (int tile = first; tile < n_tiles; tile += stride, ++it) {
    const NfTileDesc& d = S.desc[it & 3];
    const bool have_next = tile + stride < n_tiles;
    int32_t dword = 0;                       // descriptor of tile it+3 (stored at the end of the iteration)
    const bool fetch3 = tid < 16 && (long long)tile + 3ll * stride < n_tiles;
    if (fetch3) dword = __ldg(reinterpret_cast<const int32_t*>(&desc[tile + 3 * stride]) + tid);
    const float2 c = c_next;
    if (have_next) {
      const NfTileDesc& dn = S.desc[(it + 1) & 3];
      if (tid < dn.n) c_next = __ldg(&syz[dn.p0 + tid]);
    }
    const int r = d.rsf & 0xff, flag = d.rsf >> 16, n = d.n;
    const NfConst& kc = tab.row[r];
    const float4 g = kc.g;
    int* hist = S.hist[it & 1];
    int* cnt = S.cnt[it & 1];
    // wait for the staged runs of this tile (one barrier phase per tile)
    while (!mbar_try_wait(&S.full, (uint32_t)(it & 1))) {}
    // ---- phase A -------------------------------------------------------------------------------
    int nu = 0, nd = 0;
    bool slow = false;                         // m_*: result of the medium path (more than kNfK hits on a side)
    int32_t m_bu = -1, m_bd = -1;
    float m_best = 0.0f;
    if (tid < n && flag != NF_NOLINK) {
      uint32_t wd0, wd1, wu0, wu1;
      int td, tu;
      bool ok;
      if (flag == NF_STAGED) {
        const uint32_t* sUB = reinterpret_cast<const uint32_t*>(S.arena + 8 * (d.up.cn + d.dn.cn));
        ok = nf_runs(c, kc.dA, kc.dB, kc.dC, d.dn, sUB + d.up.bn, wd0, wd1, td);
        ok = nf_runs(c, kc.uA, kc.uB, kc.uC, d.up, sUB, wu0, wu1, tu) && ok;
      } else if (flag == NF_STAGED_C) {
        ok = nf_runs(c, kc.dA, kc.dB, kc.dC, d.dn, bin_start + d.dn.b0, wd0, wd1, td);
        ok = nf_runs(c, kc.uA, kc.uB, kc.uC, d.up, bin_start + d.up.b0, wu0, wu1, tu) && ok;
      } else {
        ok = false; wd0 = wd1 = wu0 = wu1 = 0;
      }
      if (ok) {
        nd = nf_test_runs<K>(c, wd0, wd1, sArena + 8u * (uint32_t)d.up.cn, kc.dA.x, kc.dA.y, -g.x, sVecD + 8u * tid, sIdxD + 2u * tid);
        nu = nf_test_runs<K>(c, wu0, wu1, sArena, kc.uA.x, kc.uA.y, g.y, sVecU + 8u * tid, sIdxU + 2u * tid);
      }
      if (ok && (nd > K || nu > K)) {               // dense region: decide now, while the staged runs are here
        int iu, id;
        if (nf_medium(c, wu0, wu1, wd0, wd1, sArena, sArena + 8u * (uint32_t)d.up.cn, kc.uA, kc.dA, g, m_best, iu, id)) {
          if (iu >= 0) { m_bu = iu + d.up.c0; m_bd = id + d.dn.c0; }
        } else {
          ok = false;                                       // exact tie: global slow path
        }
        nu = 0; nd = 0;
      }
      slow = !ok;
      if (slow) { nu = 0; nd = 0; }
      if (nu > 0 && nd > 0) atomicAdd(&hist[nd], nu);
    }
    __syncthreads();                                          // (1) phase A done: staging buffer free, histogram complete
    if (tid == 0 && have_next) issue(S.desc[(it + 1) & 3]);
    // ---- phase B1: emit one work item per up-side hit, counting-sorted by nd (descending) -------------
    int n_items = 0;
    {
      int above = 0;                                          // items with a larger nd than this thread's
#pragma unroll
      for (int k = K; k >= 1; --k) {
        const int h = hist[k];
        if (k > nd) above += h;
        n_items += h;
      }
      if (nu > 0 && nd > 0) {
        const int slot = above + atomicAdd(&cnt[nd], nu);
        const uint32_t code = (uint32_t)tid | (uint32_t)nd << 12;
#pragma unroll 1
        for (int k = 0; k < nu; ++k) S.items[slot + k] = (uint16_t)(code | (uint32_t)k << 8);
      }
    }
    __syncthreads();                                          // (2) work items complete
    if (tid < 16) { S.hist[(it + 1) & 1][tid] = 0; S.cnt[(it + 1) & 1][tid] = 0; }   // rows of the next tile
    // ---- phase B2: thread i scores item i: one up-side hit against the nd down-side hits ---------------
#pragma unroll 1
    for (int i = tid; i < n_items; i += kNfThreads) {
      const uint32_t item = S.items[i];
      const uint32_t col = 8u * (item & 255u);
      const uint32_t pa = sVecU + ((item >> 8) & 15u) * kVecRow + col;
      const int ndd = (int)(item >> 12);
      const float2 a = lds_f2(pa);
      uint32_t pb = sVecD + col;
      float best = __int_as_float(0x7f800000);
      int bid = 0, tie = 0;
#pragma unroll 1
      for (int k = 0; k < ndd; ++k, pb += kVecRow) {
        const float2 b = lds_f2(pb);
        const float ay = __fsub_rn(a.x, b.x), az = __fsub_rn(a.y, b.y);
        const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
        if (sc == best) tie = 256;
        if (sc < best) { best = sc; bid = k; }
      }
      sts_f2(pa, best, __int_as_float(bid | tie));           // the hit's vector is consumed: reuse its slot
    }
    __syncthreads();                                          // (3) item results complete
    // ---- phase C: minimum over the cluster's items, cut, stores -----------------------------------------
    if (tid < n) {
      int32_t bu = m_bu, bd = m_bd;
      float best = m_best;
      if (nu > 0 && nd > 0) {
        best = __int_as_float(0x7f800000);
        int bk = 0, bcode = 0, tie = 0;
        uint32_t pr = sVecU + 8u * tid;
#pragma unroll 1
        for (int k = 0; k < nu; ++k, pr += kVecRow) {
          const float2 res = lds_f2(pr);
          const int code = __float_as_int(res.y);
          if (res.x == best) tie = 256;
          if (res.x < best) { best = res.x; bk = k; bcode = code; }
          tie |= code & 256;
        }
        if (tie) slow = true;
        else {
          bu = (int32_t)lds_u16(sIdxU + (uint32_t)bk * kIdxRow + 2u * tid) + d.up.c0;
          bd = (int32_t)lds_u16(sIdxD + (uint32_t)(bcode & 255) * kIdxRow + 2u * tid) + d.dn.c0;
        }
      }
      if (slow) {
        const int s = (d.rsf >> 8) & 0xff;
        nf_slow(c, kc, bin_start + (size_t)s * nbp1, syz + d.sec_off, order + d.sec_off, best, bu, bd);
      }
      if (!(bu >= 0 && best <= g.z)) { bu = -1; bd = -1; }
      link_up[d.p0 + tid] = bu;
      link_dn[d.p0 + tid] = bd;
    }
    if (fetch3) reinterpret_cast<int32_t*>(&S.desc[(it + 3) & 3])[tid] = dword;
    // no barrier here: phase A of the next tile writes only the thread's own cache column, the other
    // histogram row and (after its mbarrier wait) reads the staging buffer refilled after barrier (1).
  }
}

// ---- K3: link cleaner + per-tile start-hit count -------------------------
// up'[c] = (up[c] = u >= 0 and dn[u] = c) ? u : -1;  dn'[c] likewise; out of place.
// Tile = 2048 clusters (256 threads x 8, strided for coalescing); tiles never cross a sector.
__global__ void __launch_bounds__(256)
k_clean_links(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
              const int32_t* __restrict__ up_raw, const int32_t* __restrict__ dn_raw,
              int32_t* __restrict__ up, int32_t* __restrict__ dn, int2* __restrict__ tile_cnt,
              uint32_t* __restrict__ start_bits /*[tile][64]: bit p of the tile = start hit (read by S4)*/,
              const DevStatus* __restrict__ st) {
  __shared__ int ws[33];
  if (st->err_range) {     // S1 dropped clusters (row >= n_rows): positions >= n - dropped were never written by S1 / S2.
    // The run is reported as TPCCA_E_RANGE; S3-S5 produce nothing (no start hit) instead of following stale links.
    if (threadIdx.x < 64) start_bits[(size_t)blockIdx.x * 64 + threadIdx.x] = 0u;
    if (threadIdx.x == 0) tile_cnt[blockIdx.x] = make_int2(0, 0);
    return;
  }
  const int ns = __ldg(&T->n_sectors);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].tile2048); });
  const int n = __ldg(&sec[s].n), off = __ldg(&sec[s].off);
  const int p0 = (blockIdx.x - __ldg(&sec[s].tile2048)) * 2048;
  int cnt = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int p = p0 + k * 256 + threadIdx.x;
    bool is_start = false;
    if (p < n) {
      const int32_t u = up_raw[off + p], d = dn_raw[off + p];
      // (u, d < n always holds for links written by S2; the bound is a safety net against stale workspace bytes)
      const int32_t uc = (u >= 0 && u < n && __ldg(&dn_raw[off + u]) == p) ? u : -1;
      const int32_t dc = (d >= 0 && d < n && __ldg(&up_raw[off + d]) == p) ? d : -1;
      up[off + p] = uc;
      dn[off + p] = dc;
      is_start = (dc == -1 && uc >= 0);
      cnt += is_start ? 1 : 0;
    }
    // the 32 positions of a warp are consecutive: one ballot = one word of the tile's start-hit bitmap
    const unsigned m = __ballot_sync(0xffffffffu, is_start);
    if ((threadIdx.x & 31) == 0) start_bits[(size_t)blockIdx.x * 64 + k * 8 + (threadIdx.x >> 5)] = m;
  }
  int total;
  block_exclusive_scan<int>(cnt, ws, total);
  if (threadIdx.x == 0) tile_cnt[blockIdx.x] = make_int2(total, 0);
}

// ---- generic single-block exclusive scan over per-tile (a, b) pairs ---------------------------
// out[t] = sum of in[0..t); totals to tot[0], tot[1].  In place allowed.
__global__ void __launch_bounds__(1024)
k_scan_pairs(const int2* __restrict__ in, longlong2* __restrict__ out, int n_tiles, int64_t* __restrict__ tot) {
  __shared__ long long ws[33];
  long long ca = 0, cb = 0;
  for (int base = 0; base < n_tiles; base += 1024) {
    const int t = base + threadIdx.x;
    const int2 v = t < n_tiles ? in[t] : make_int2(0, 0);
    long long ta, tb;
    const long long ea = block_exclusive_scan<long long>((long long)v.x, ws, ta);
    const long long eb = block_exclusive_scan<long long>((long long)v.y, ws, tb);
    if (t < n_tiles) out[t] = make_longlong2(ca + ea, cb + eb);
    ca += ta; cb += tb;
  }
  if (threadIdx.x == 0) { tot[0] = ca; tot[1] = cb; }
}

// ---- K4a: after the tile scan: sector start offsets, total, capacity check ---------------------
__global__ void k_start_offsets(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
                                const longlong2* __restrict__ tile_off, const int64_t* __restrict__ tot,
                                int n_tiles, int32_t cap, DevStatus* __restrict__ st) {
  const int ns = T->n_sectors;
  const int s = threadIdx.x;
  if (s <= ns) {
    const int t = sec[s].tile2048;     // sec[ns].tile2048 = n_tiles
    st->start_off[s] = (int32_t)(t < n_tiles ? tile_off[t].x : tot[0]);
  }
  if (s == 0) {
    st->n_start = (int32_t)tot[0];
    if (tot[0] > (int64_t)cap) st->err_capacity = 1;
    for (int i = 0; i < 8; ++i) st->work_counter[i] = 0;
  }
}

// ---- K4b: ordered compaction of the start hits ---------------------------------
// Each thread owns 8 CONSECUTIVE positions so that ranks are ascending in sorted position.
__global__ void __launch_bounds__(256)
k_start_hits(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
             const uint32_t* __restrict__ start_bits,
             const longlong2* __restrict__ tile_off, int32_t cap, int32_t* __restrict__ start_hit) {
  __shared__ int ws[33];
  const int ns = __ldg(&T->n_sectors);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].tile2048); });
  const int p0 = (blockIdx.x - __ldg(&sec[s].tile2048)) * 2048 + threadIdx.x * 8;
  // the thread's 8 consecutive positions are one byte of the bitmap S3 wrote (positions >= n hold 0 bits)
  const unsigned flags = (__ldg(&start_bits[(size_t)blockIdx.x * 64 + (threadIdx.x >> 2)]) >> ((threadIdx.x & 3) * 8)) & 0xffu;
  int total;
  int rank = block_exclusive_scan<int>(__popc(flags), ws, total);
  long long o = tile_off[blockIdx.x].x + rank;
#pragma unroll
  for (int k = 0; k < 8; ++k)
    if (flags & (1u << k)) {
      if (o < cap) start_hit[o] = p0 + k;
      ++o;
    }
}

// ---- K4c-e: processing order of S5 ---------------------------------------------------
// Tracks are emitted in start-hit order, but the ORDER IN WHICH S5 works through the start hits is
// free.  Walking them sector by sector in ascending z (time) instead of row-major keeps the clusters
// and bin_start entries touched by the tracklets in flight inside a z window of the sector, i.e. in
// L2.  The unit of the ordering is the S1 coarse bucket (row, z slab): its start hits are one
// contiguous range of slots; zorder[j] = j-th bucket of a sector by ascending z (host table).
__global__ void __launch_bounds__(256)
k_sh_bucket_counts(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, const int32_t* __restrict__ zorder,
                   const uint32_t* __restrict__ cb_start, const int32_t* __restrict__ start_hit, int32_t cap,
                   int32_t* __restrict__ sh_first, int32_t* __restrict__ cnt, int2* __restrict__ blk_cnt) {
  __shared__ int ws[33];
  const int ncb = T->n_cb, ns = T->n_sectors;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  int a = 0, n = 0;
  if (i < ns * ncb && !st->err_capacity) {
    const int s = i / ncb, j = i - s * ncb;
    const int cb = zorder[j];
    const uint32_t lo_pos = cb_start[(size_t)s * (ncb + 1) + cb], hi_pos = cb_start[(size_t)s * (ncb + 1) + cb + 1];
    const int s0 = st->start_off[s], s1 = st->start_off[s + 1];
    auto lower = [&](uint32_t pos) {             // first slot in [s0, s1) whose start hit is >= pos
      int lo = s0, hi = s1;
      while (lo < hi) { const int mid = (lo + hi) >> 1; if ((uint32_t)start_hit[mid] < pos) lo = mid + 1; else hi = mid; }
      return lo;
    };
    a = lower(lo_pos);
    n = lower(hi_pos) - a;
  }
  if (i < ns * ncb) { sh_first[i] = a; cnt[i] = n; }
  int total;
  block_exclusive_scan<int>(n, ws, total);
  if (threadIdx.x == 0) blk_cnt[blockIdx.x] = make_int2(total, 0);
}

// perm[j] = work record of the j-th tracklet in processing order: (slot, start row | sector << 16, start hit, 0).
// One 16-byte load gives the S5 kernels everything a refill needs (no row / sector search, no second
// dependent load of start_hit): the row of a bucket's start hits is the bucket's row.
__global__ void __launch_bounds__(256)
k_sh_perm(const DevTables* __restrict__ T, const int32_t* __restrict__ zorder, const int32_t* __restrict__ start_hit,
          const int32_t* __restrict__ sh_first, const int32_t* __restrict__ cnt,
          const longlong2* __restrict__ blk_pre, int4* __restrict__ perm) {
  __shared__ int ws[33];
  const int ncb = T->n_cb;
  const int n = T->n_sectors * ncb;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int c = i < n ? cnt[i] : 0;
  int total;
  const int ex = block_exclusive_scan<int>(c, ws, total);
  if (i >= n || c == 0) return;
  const int s = i / ncb, j = i - s * ncb;
  int r, k;
  cb_row_slab(T, zorder[j], r, k);
  const int a = sh_first[i];
  int4* o = perm + blk_pre[blockIdx.x].x + ex;
  for (int q = 0; q < c; ++q) o[q] = make_int4(a + q, r | (s << 16), start_hit[a + q], 0);
}

}  // namespace tpcca
