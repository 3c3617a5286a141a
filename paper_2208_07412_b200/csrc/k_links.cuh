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
#ifndef TPCCA_NF_K
#define TPCCA_NF_K 8
#endif
#ifndef TPCCA_NF_CAPC
#define TPCCA_NF_CAPC 512
#endif
#ifndef TPCCA_NF_CAPB
#define TPCCA_NF_CAPB 2048
#endif
constexpr int kNfK = TPCCA_NF_K;          // window hits cached per side and thread in shared memory
constexpr int kNfThreads = kNfTile;       // one thread per cluster of the tile
constexpr int kNfCapC = TPCCA_NF_CAPC;    // staged clusters per side (8 B each)
constexpr int kNfCapB = TPCCA_NF_CAPB;    // staged bin_start entries per side (4 B each)

#ifdef TPCCA_NF_STATS
__device__ unsigned long long g_nf_hist[4][64];   // tests per side, hits per side, pairs, pairs under cut
#endif
enum { NF_STAGED = 0, NF_NOLINK = 1, NF_GLOBAL = 2 };

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
  if (cn > kNfCapC || bn > kNfCapB || (s_hi - s_lo) >= (1 << 24)) flag = NF_GLOBAL;
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
      }
      d.rsf = r | (s << 8) | (flag << 16);
      desc[t] = d;
    }
  }
}

// ---- candidate gathering ---------------------------------------------------------------------------
// Window candidates of one side (A, B, C = the side's NfConst groups): every cluster q of the
// neighbour row with |y_q - y_c| <= hy and |z_q - z_c| <= hz.  The bin range is a superset of the
// window; the z slices of the range are walked as ONE flattened loop so that the
// lanes of a warp, whose slices hold different numbers of clusters, stay together.
// Caches (dy * dxo, dz * dxo) and the position of the first kNfK hits; returns the number of hits.
// UP: the cached vector is (y_q - y_c) * dxo; down side: (y_c - y_q) * dxo (fl(a - b) = -fl(b - a),
// so the negation is exact).
struct NfCache {
  float2 uv[kNfK][kNfThreads];
  float2 dv[kNfK][kNfThreads];
  int32_t ui[kNfK][kNfThreads];
  int32_t di[kNfK][kNfThreads];
};

// global-memory version (tiles whose neighbour runs do not fit the staging buffers)
template <bool UP>
__device__ __forceinline__ int nf_gather(const float2 c, const float4 A, const float4 B, const int4 C, const float dxo,
                                         const uint32_t* __restrict__ bs,
                                         const float2* __restrict__ yz, float2 (*s_v)[kNfThreads],
                                         int32_t (*s_i)[kNfThreads], const int tid) {
  const int by0 = bin_range(__fsub_rn(c.x, A.z), B.x, B.y, C.x), by1 = bin_range(__fadd_rn(c.x, A.z), B.x, B.y, C.x);
  const int bz0 = bin_range(__fsub_rn(c.y, A.w), B.w, B.z, C.y), bz1 = bin_range(__fadd_rn(c.y, A.w), B.w, B.z, C.y);
  const uint32_t* bp = bs + C.w + bz0 * C.z;
  const int nsl = bz1 - bz0 + 1;
  uint32_t q = __ldg(&bp[by0]), e = __ldg(&bp[by1 + 1]);
  uint32_t q1 = 0, e1 = 0;
  if (nsl > 1) { q1 = __ldg(&bp[C.z + by0]); e1 = __ldg(&bp[C.z + by1 + 1]); }
  int k = 0, n = 0;
  for (;;) {
    if (q >= e) {
      if (++k >= nsl) break;
      if (k == 1) { q = q1; e = e1; }
      else { q = __ldg(&bp[k * C.z + by0]); e = __ldg(&bp[k * C.z + by1 + 1]); }
      continue;
    }
    const float2 v = __ldg(&yz[q]);
    const float dy = __fsub_rn(v.x, c.x), dz = __fsub_rn(v.y, c.y);
    if (fabsf(dy) <= A.x && fabsf(dz) <= A.y) {
      if (n < kNfK) {
        s_v[n][tid] = make_float2(__fmul_rn(UP ? dy : -dy, dxo), __fmul_rn(UP ? dz : -dz, dxo));
        s_i[n][tid] = (int32_t)q;
      }
      ++n;
    }
    ++q;
  }
  return n;
}

// shared-memory version: sC / sB are the staged cluster / bin_start runs of the side.  Returns the
// number of hits, or -1 if the cluster's slices are not covered by the staged range (the caller then
// takes the global-memory path for this cluster).
template <bool UP>
__device__ __forceinline__ int nf_gather_smem(const float2 c, const float4 A, const float4 B, const int4 C, const float dxo,
                                              const NfSide& sd, const float2* __restrict__ sC,
                                              const uint32_t* __restrict__ sB, float2 (*s_v)[kNfThreads],
                                              int32_t (*s_i)[kNfThreads], const int tid) {
  const int by0 = bin_range(__fsub_rn(c.x, A.z), B.x, B.y, C.x), by1 = bin_range(__fadd_rn(c.x, A.z), B.x, B.y, C.x);
  const int bz0 = bin_range(__fsub_rn(c.y, A.w), B.w, B.z, C.y), bz1 = bin_range(__fadd_rn(c.y, A.w), B.w, B.z, C.y);
  const int ds = sd.ds_shift & 0xffffff, shift = sd.ds_shift >> 24;
  const int k0 = bz0 - sd.s0;
  if (k0 < 0 || bz1 - sd.s0 > ds) return -1;
  const uint32_t* bp = sB + shift + k0 * C.z;
  int n = 0;
  // two slices per pass (a window spans two slices, three when it straddles a bin edge by < margin)
  for (int ks = bz1 - bz0; ks >= 0; ks -= 2, bp += 2 * C.z) {
    const int q = (int)bp[by0] - sd.c0;
    const int n0 = (int)bp[by1 + 1] - sd.c0 - q;
    int total = n0, o1 = 0;
    if (ks > 0) {
      const int q1 = (int)bp[C.z + by0] - sd.c0;
      total += (int)bp[C.z + by1 + 1] - sd.c0 - q1;
      o1 = q1 - q - n0;                    // flat index j >= n0 -> staged index q + j + o1
    }
#ifdef TPCCA_NF_STATS
    atomicAdd(&g_nf_hist[0][min(total, 63)], 1ull);
#endif
    for (int j = 0; j < total; ++j) {
      const int idx = q + j + (j >= n0 ? o1 : 0);
      const float2 v = sC[idx];
      const float dy = __fsub_rn(v.x, c.x), dz = __fsub_rn(v.y, c.y);
      if (fabsf(dy) <= A.x && fabsf(dz) <= A.y) {
        if (n < kNfK) {
          s_v[n][tid] = make_float2(__fmul_rn(UP ? dy : -dy, dxo), __fmul_rn(UP ? dz : -dz, dxo));
          s_i[n][tid] = idx + sd.c0;
        }
        ++n;
      }
    }
  }
  return n;
}

// visit every window candidate of one side (plain nested loops; slow path only)
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
// id): the full U x D product by nested rescans of both windows.
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

// best pair over the cached hits (nu, nd <= kNfK).  Returns false on an exact score tie (decided by
// original ids in the slow path).
__device__ __forceinline__ bool nf_best_pair(const NfCache& ch, int tid, int nu, int nd, float& best, int32_t& bu, int32_t& bd) {
  const int np = nu * nd;
  int iu = 0, id = 0, bi = 0, bj = 0;
  bool tie = false;
  best = __int_as_float(0x7f800000);
  for (int k = 0; k < np; ++k) {
    const float2 a = ch.uv[iu][tid], b = ch.dv[id][tid];
    const float ay = __fsub_rn(a.x, b.x), az = __fsub_rn(a.y, b.y);
    const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
    tie |= (sc == best);
    if (sc < best) { best = sc; bi = iu; bj = id; }
    if (++id == nd) { id = 0; ++iu; }
  }
  bu = -1; bd = -1;
  if (np > 0) { bu = ch.ui[bi][tid]; bd = ch.di[bj][tid]; }
  return !tie;
}

struct NfStage {
  float2 uc[kNfCapC];
  float2 dc[kNfCapC];
  uint32_t ub[kNfCapB];
  uint32_t db[kNfCapB];
};
struct NfSmem {
  NfStage st[2];
  NfCache ch;
  NfTileDesc desc[4];
  uint64_t full[2];
};

// ---- K2b: neighbour finder, one thread per cluster --------------------------
// For cluster c of row r (1 <= r <= n_rows-2): over U x D (exact windows in rows r+1, r-1) the
// pair minimising score = ay^2 + az^2, ay = (yu-yc)*dxd - (yc-yd)*dxu; ties -> smallest original
// id of u, then of d; stored if score <= nf_cut[r].
// Persistent blocks walk the tile list with a grid stride (so the tiles in flight are neighbours in
// memory and the three-fold reuse of a row stays in L2).  Iteration i: thread 0 issues the bulk
// copies of tile i+1 into stage (i+1)&1, warp 0 fetches the descriptor of tile i+3, every thread
// prefetches its own cluster of tile i+1, then the block waits for stage i&1 and searches tile i in
// shared memory.  Per-row constants come from the constant bank (NfTable is a kernel parameter).
__global__ void __launch_bounds__(kNfThreads)
k_neighbours(const __grid_constant__ NfTable tab, const float2* __restrict__ syz,
             const uint32_t* __restrict__ bin_start, const int32_t* __restrict__ order, uint32_t nbp1,
             const int32_t* __restrict__ n_tiles_ptr, const NfTileDesc* __restrict__ desc,
             int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  extern __shared__ __align__(128) unsigned char nf_smem_raw[];
  NfSmem& S = *reinterpret_cast<NfSmem*>(nf_smem_raw);
  const int tid = threadIdx.x;
  const int n_tiles = __ldg(n_tiles_ptr);
  const int stride = gridDim.x;
  const int first = blockIdx.x;
  if (first >= n_tiles) return;
  if (tid == 0) { mbar_init(&S.full[0], 1); mbar_init(&S.full[1], 1); fence_mbar_init(); }
  // descriptors of the block's first three tiles
  if (tid < 48) {
    const int k = tid >> 4, t = first + k * stride;
    if (t < n_tiles) reinterpret_cast<int32_t*>(&S.desc[k])[tid & 15] = __ldg(reinterpret_cast<const int32_t*>(&desc[t]) + (tid & 15));
  }
  __syncthreads();
  auto issue = [&](const NfTileDesc& d, int stage) {      // thread 0 only
    uint32_t bytes = 0;
    const bool staged = (d.rsf >> 16) == NF_STAGED;
    if (staged) bytes = 8u * (uint32_t)(d.up.cn + d.dn.cn) + 4u * (uint32_t)(d.up.bn + d.dn.bn);
    mbar_arrive_expect_tx(&S.full[stage], bytes);
    if (staged) {
      NfStage& st = S.st[stage];
      if (d.up.cn) bulk_g2s(st.uc, syz + (d.sec_off + d.up.c0), 8u * d.up.cn, &S.full[stage]);
      if (d.dn.cn) bulk_g2s(st.dc, syz + (d.sec_off + d.dn.c0), 8u * d.dn.cn, &S.full[stage]);
      if (d.up.bn) bulk_g2s(st.ub, bin_start + d.up.b0, 4u * d.up.bn, &S.full[stage]);
      if (d.dn.bn) bulk_g2s(st.db, bin_start + d.dn.b0, 4u * d.dn.bn, &S.full[stage]);
    }
  };
  if (tid == 0) issue(S.desc[0], 0);
  float2 c_next = make_float2(0.f, 0.f);
  if (tid < S.desc[0].n) c_next = __ldg(&syz[S.desc[0].p0 + tid]);
  int it = 0;
  for (int tile = first; tile < n_tiles; tile += stride, ++it) {
    const int stage = it & 1;
    const NfTileDesc& d = S.desc[it & 3];
    const bool have_next = tile + stride < n_tiles;
    // descriptor of tile it+3 -> registers of warp 0 (stored at the end of the iteration)
    int32_t dword = 0;
    const bool fetch3 = tid < 16 && (long long)tile + 3ll * stride < n_tiles;
    if (fetch3) dword = __ldg(reinterpret_cast<const int32_t*>(&desc[tile + 3 * stride]) + tid);
    if (tid == 0 && have_next) issue(S.desc[(it + 1) & 3], stage ^ 1);
    const float2 c = c_next;
    if (have_next) {
      const NfTileDesc& dn = S.desc[(it + 1) & 3];
      if (tid < dn.n) c_next = __ldg(&syz[dn.p0 + tid]);
    }
    const int r = d.rsf & 0xff, flag = d.rsf >> 16;
    const bool active = tid < d.n;
    // wait for the staged runs of this tile (phase parity of the stage's barrier = (it >> 1) & 1)
    while (!mbar_try_wait(&S.full[stage], (uint32_t)((it >> 1) & 1))) {}
    int32_t bu = -1, bd = -1;
    if (active && flag != NF_NOLINK) {
      const NfConst& kc = tab.row[r];
      const float4 g = kc.g;
      float best = 0.0f;
      int nd, nu;
      if (flag == NF_STAGED) {
        const NfStage& st = S.st[stage];
        nd = nf_gather_smem<false>(c, kc.dA, kc.dB, kc.dC, g.x, d.dn, st.dc, st.db, S.ch.dv, S.ch.di, tid);
        nu = nf_gather_smem<true>(c, kc.uA, kc.uB, kc.uC, g.y, d.up, st.uc, st.ub, S.ch.uv, S.ch.ui, tid);
      } else {
        const int s = (d.rsf >> 8) & 0xff;
        const uint32_t* bs = bin_start + (size_t)s * nbp1;
        const float2* yz = syz + d.sec_off;
        nd = nf_gather<false>(c, kc.dA, kc.dB, kc.dC, g.x, bs, yz, S.ch.dv, S.ch.di, tid);
        nu = nf_gather<true>(c, kc.uA, kc.uB, kc.uC, g.y, bs, yz, S.ch.uv, S.ch.ui, tid);
      }
#ifdef TPCCA_NF_STATS
      atomicAdd(&g_nf_hist[1][min(max(nd, 0), 63)], 1ull);
      atomicAdd(&g_nf_hist[1][min(max(nu, 0), 63)], 1ull);
      atomicAdd(&g_nf_hist[2][min(max(nu * nd, 0), 63)], 1ull);
#endif
      bool done = false;
      if (nd >= 0 && nu >= 0 && nd <= kNfK && nu <= kNfK) done = nf_best_pair(S.ch, tid, nu, nd, best, bu, bd);
      if (!done) {
        const int s = (d.rsf >> 8) & 0xff;
        nf_slow(c, kc, bin_start + (size_t)s * nbp1, syz + d.sec_off, order + d.sec_off, best, bu, bd);
      }
      if (!(bu >= 0 && best <= g.z)) { bu = -1; bd = -1; }
    }
    if (active) {
      link_up[d.p0 + tid] = bu;
      link_dn[d.p0 + tid] = bd;
    }
    __syncthreads();           // stage and descriptor slot are free again
    if (fetch3) reinterpret_cast<int32_t*>(&S.desc[(it + 3) & 3])[tid] = dword;
    // (visible to every thread after the next iteration's __syncthreads; it is first read two iterations later)
  }
}

// ---- K3: link cleaner + per-tile start-hit count -------------------------
// up'[c] = (up[c] = u >= 0 and dn[u] = c) ? u : -1;  dn'[c] likewise; out of place.
// Tile = 2048 clusters (256 threads x 8, strided for coalescing); tiles never cross a sector.
__global__ void __launch_bounds__(256)
k_clean_links(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
              const int32_t* __restrict__ up_raw, const int32_t* __restrict__ dn_raw,
              int32_t* __restrict__ up, int32_t* __restrict__ dn, int2* __restrict__ tile_cnt) {
  __shared__ int ws[33];
  const int ns = __ldg(&T->n_sectors);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].tile2048); });
  const int n = __ldg(&sec[s].n), off = __ldg(&sec[s].off);
  const int p0 = (blockIdx.x - __ldg(&sec[s].tile2048)) * 2048;
  int cnt = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int p = p0 + k * 256 + threadIdx.x;
    if (p < n) {
      const int32_t u = up_raw[off + p], d = dn_raw[off + p];
      const int32_t uc = (u >= 0 && __ldg(&dn_raw[off + u]) == p) ? u : -1;
      const int32_t dc = (d >= 0 && __ldg(&up_raw[off + d]) == p) ? d : -1;
      up[off + p] = uc;
      dn[off + p] = dc;
      cnt += (dc == -1 && uc >= 0) ? 1 : 0;
    }
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
    st->work_counter = 0;
  }
}

// ---- K4b: ordered compaction of the start hits ---------------------------------
// Each thread owns 8 CONSECUTIVE positions so that ranks are ascending in sorted position.
__global__ void __launch_bounds__(256)
k_start_hits(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
             const int32_t* __restrict__ up, const int32_t* __restrict__ dn,
             const longlong2* __restrict__ tile_off, int32_t cap, int32_t* __restrict__ start_hit) {
  __shared__ int ws[33];
  const int ns = __ldg(&T->n_sectors);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].tile2048); });
  const int n = __ldg(&sec[s].n), off = __ldg(&sec[s].off);
  const int p0 = (blockIdx.x - __ldg(&sec[s].tile2048)) * 2048 + threadIdx.x * 8;
  unsigned flags = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int p = p0 + k;
    if (p < n && dn[off + p] == -1 && up[off + p] >= 0) flags |= 1u << k;
  }
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

}  // namespace tpcca
