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
// of sorted clusters: the z slices S_lo..S_hi of that row.  k_nf_plan writes one descriptor per tile;
// k_neighbours stages the two cluster runs of the NEXT tile in shared memory with 1-D bulk async
// copies (TMA, mbarrier completion, two buffers) while the current tile is searched in shared memory.
// bin_start is not read at all on the fast path: the first staged cluster of every z slice is found
// from the staged clusters themselves (a z slice of a row holds ~5 clusters at the headline density, so
// walking the whole slices of a window costs about as much as looking the y bins up, without the loads).
#ifndef TPCCA_NF_K
#define TPCCA_NF_K 12
#endif
constexpr int kNfK = TPCCA_NF_K;          // window hits listed per side and thread in shared memory
constexpr int kNfThreads = kNfTile;       // one thread per cluster of the tile
constexpr int kNfArenaC = 768;            // staged clusters per buffer (both sides together)
constexpr int kNfMaxSl = 254;             // z slices per side whose first cluster is indexed

enum { NF_STAGED = 0, NF_NOLINK = 1, NF_GLOBAL = 2 };

struct NfSide {        // staging of one neighbour row for one tile
  int32_t c0;          // sector-local sorted position of staged cluster 0 ((sec_off + c0) is even; may be -1)
  int32_t cn;          // staged clusters (even)
  int32_t s0;          // first staged z slice
  int32_t nsl;         // staged z slices
  int32_t lo, hi;      // staged indices [lo, hi) are the clusters of slices s0 .. s0 + nsl - 1 (the rest is alignment)
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
  const uint32_t gb_hi = bs_off + (uint32_t)(T->bin_base[rn] + (s_hi + 1) * ny);   // end of slice s_hi
  const int c_lo = (int)bin_start[gb_lo], c_hi = (int)bin_start[gb_hi];
  const int c0 = c_lo - ((sec_off + c_lo) & 1);
  const int cn = (c_hi - c0 + 1) & ~1;
  o.c0 = c0; o.cn = cn; o.s0 = s_lo; o.nsl = s_hi - s_lo + 1; o.lo = c_lo - c0; o.hi = c_hi - c0;
  if (o.nsl > kNfMaxSl) flag = NF_GLOBAL;
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
      d.up = NfSide{0, 0, 0, 0, 0, 0};
      d.dn = d.up;
      if (!edge) {
        const int b_first = bin_range(syz[d.p0].y, zlo, ibz, nz_r - 1);
        const int b_last = bin_range(syz[d.p0 + d.n - 1].y, zlo, ibz, nz_r - 1);
        nf_plan_side(d.up, flag, T, r + 1, T->hz_up[r] + T->margin, b_first, b_last, nz_r, bin_r, bs_off, sec_off, bin_start);
        nf_plan_side(d.dn, flag, T, r - 1, T->hz_dn[r] + T->margin, b_first, b_last, nz_r, bin_r, bs_off, sec_off, bin_start);
        if (d.up.cn + d.dn.cn > kNfArenaC) flag = NF_GLOBAL;
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
// are not covered by the staged runs or whose best score is tied.
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

// ---- shared-memory accessors on 32-bit shared addresses (no 64-bit pointer arithmetic in the loops) --
__device__ __forceinline__ float2 lds_f2(uint32_t a) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ float lds_f1(uint32_t a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
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

constexpr uint32_t kVecRow = 8u * kNfThreads;   // bytes between consecutive rows of the down-vector cache
constexpr uint32_t kIdxRow = 2u * kNfThreads;   // ... of the hit lists

template <int K>
struct NfSmem {
  alignas(128) float2 arena[2][kNfArenaC];   // two staging buffers (TMA destinations): [up clusters | down clusters]
  float2 vecD[K][kNfThreads];                // (y_d - y_c, z_d - z_c) * (-dxu) of the listed down-side hits; column = cluster
  uint16_t list[2][K][kNfThreads];           // staged indices of the window hits: [0] down side, [1] up side
  uint16_t sidx[2][2][kNfMaxSl + 2];         // [buffer][side]: first staged index of every staged z slice (+ end)
  NfTileDesc desc[4];
  uint64_t full[2];
};

// ---- phase 0: first staged index of every z slice of one side --------------------------------------
// The staged run [lo, hi) holds the clusters of slices s0 .. s0 + nsl - 1 in slice order.  sidx[k] = first
// index whose slice is >= s0 + k (k = 0 .. nsl; sidx[nsl] = hi): every thread looks at a few staged clusters
// and, where the slice changes, fills the entries of the slices that start there.
__device__ __forceinline__ void nf_slice_index(const NfSide& sd, uint32_t sA, float zlo, float ibz, int nzh,
                                               uint16_t* __restrict__ sidx, int tid) {
  const int lo = sd.lo, hi = sd.hi, nsl = sd.nsl;
  if (lo >= hi) {
    for (int k = tid; k <= nsl; k += kNfThreads) sidx[k] = (uint16_t)lo;
    return;
  }
  for (int i = lo + tid; i < hi; i += kNfThreads) {
    const int b = min(max(bin_range(lds_f1(sA + 8u * (uint32_t)i + 4u), zlo, ibz, nzh) - sd.s0, 0), nsl - 1);
    const int bp = (i == lo) ? -1 : min(max(bin_range(lds_f1(sA + 8u * (uint32_t)i - 4u), zlo, ibz, nzh) - sd.s0, 0), nsl - 1);
    for (int k = bp + 1; k <= b; ++k) sidx[k] = (uint16_t)i;
    if (i == hi - 1)
      for (int k = b + 1; k <= nsl; ++k) sidx[k] = (uint16_t)hi;
  }
}

// ---- phase A: window test of the staged run [j0, j1) of one side -------------------------------------
// Hits (staged indices) go to the thread's list column at pl + k * kIdxRow; returns the number of hits
// (may exceed K; only the first K are listed).
template <int K>
__device__ __forceinline__ int nf_test_run(const float2 c, uint32_t sA, int j0, int j1, float hy, float hz, uint32_t pl) {
  int n = 0;
  uint32_t a = sA + 8u * (uint32_t)j0;
  const uint32_t e = sA + 8u * (uint32_t)j1;
#pragma unroll 2
  for (; a < e; a += 8u) {
    const float2 v = lds_f2(a);
    const float dy = __fsub_rn(v.x, c.x), dz = __fsub_rn(v.y, c.y);
    if (fabsf(dy) <= hy && fabsf(dz) <= hz) {
      if (n < K) sts_u16(pl + (uint32_t)n * kIdxRow, (a - sA) >> 3);
      ++n;
    }
  }
  return n;
}

// ---- medium path: more than K hits on a side (dense regions) -----------------------------------------
// Nested loops over the staged candidate runs of both sides (no lists): the U x D product in the order
// and arithmetic of nf_slow, in shared memory.  Returns false on an exact score tie (decided by original
// ids in nf_slow).  iu / id are staged indices.
__device__ __noinline__ bool nf_medium(const float2 c, uint32_t sAU, int ju0, int ju1, uint32_t sAD, int jd0, int jd1,
                                       const float4 uA, const float4 dA, const float4 g, float& best, int& iu, int& id) {
  bool have = false, tie = false;
  best = 0.0f; iu = -1; id = -1;
#pragma unroll 1
  for (int ju = ju0; ju < ju1; ++ju) {
    const float2 u = lds_f2(sAU + 8u * (uint32_t)ju);
    const float dyu = __fsub_rn(u.x, c.x), dzu = __fsub_rn(u.y, c.y);
    if (!(fabsf(dyu) <= uA.x && fabsf(dzu) <= uA.y)) continue;
    const float Ay = __fmul_rn(dyu, g.y), Az = __fmul_rn(dzu, g.y);
#pragma unroll 1
    for (int jd = jd0; jd < jd1; ++jd) {
      const float2 d = lds_f2(sAD + 8u * (uint32_t)jd);
      const float dyd = __fsub_rn(d.x, c.x), dzd = __fsub_rn(d.y, c.y);
      if (!(fabsf(dyd) <= dA.x && fabsf(dzd) <= dA.y)) continue;
      const float ay = __fsub_rn(Ay, __fmul_rn(-dyd, g.x));
      const float az = __fsub_rn(Az, __fmul_rn(-dzd, g.x));
      const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
      if (have && sc == best) tie = true;
      if (!have || sc < best) { have = true; best = sc; iu = ju; id = jd; }
    }
  }
  return !tie;
}

// ---- K2b: neighbour finder --------------------------------------------------
// For cluster c of row r (1 <= r <= n_rows-2): over U x D (exact windows in rows r+1, r-1) the
// pair minimising score = ay^2 + az^2, ay = (yu-yc)*dxd - (yc-yd)*dxu; ties -> smallest original
// id of u, then of d; stored if score <= nf_cut[r].
// Persistent blocks walk the tile list with a grid stride (tiles in flight are neighbours in memory,
// so the three-fold reuse of a row stays in L2).  Per tile, ONE block barrier:
//   phase 0  the first staged index of every z slice of both neighbour runs (from the staged clusters);
//   barrier; thread 0 issues the bulk copies of the NEXT tile into the other buffer;
//   phase A  thread t = cluster t: the z slices its two windows touch -> one contiguous staged run per
//            side (the grid is only an accelerator: every cluster of those slices gets the exact window
//            test); hits are listed in the thread's shared-memory column;
//   phase B  thread t: the nd down vectors once, then the nu x nd pair scores in the defined operation
//            order, minimum, cut, coalesced link stores.  An exact tie of the minimum goes to nf_slow.
#ifndef TPCCA_NF_BPS
#define TPCCA_NF_BPS 6
#endif
template <int K>
__global__ void __launch_bounds__(kNfThreads, TPCCA_NF_BPS)
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
  if (tid == 0) { mbar_init(&S.full[0], 1); mbar_init(&S.full[1], 1); fence_mbar_init(); }
  if (tid < 48) {      // descriptors of the block's first three tiles
    const int k = tid >> 4, t = first + k * stride;
    if (t < n_tiles) reinterpret_cast<int32_t*>(&S.desc[k])[tid & 15] = __ldg(reinterpret_cast<const int32_t*>(&desc[t]) + (tid & 15));
  }
  __syncthreads();
  auto issue = [&](const NfTileDesc& d, int buf) {      // thread 0 only
    const int flag = d.rsf >> 16;
    const uint32_t bytes = flag == NF_STAGED ? 8u * (uint32_t)(d.up.cn + d.dn.cn) : 0u;
    mbar_arrive_expect_tx(&S.full[buf], bytes);
    if (bytes) {
      float2* a = S.arena[buf];
      if (d.up.cn) bulk_g2s(a, syz + (d.sec_off + d.up.c0), 8u * d.up.cn, &S.full[buf]);
      if (d.dn.cn) bulk_g2s(a + d.up.cn, syz + (d.sec_off + d.dn.c0), 8u * d.dn.cn, &S.full[buf]);
    }
  };
  if (tid == 0) issue(S.desc[0], 0);
  float2 c_next = make_float2(0.f, 0.f);
  if (tid < S.desc[0].n) c_next = __ldg(&syz[S.desc[0].p0 + tid]);
  const uint32_t sListD = smem_u32(&S.list[0][0][0]) + 2u * tid, sListU = smem_u32(&S.list[1][0][0]) + 2u * tid;
  const uint32_t sVec = smem_u32(&S.vecD[0][0]) + 8u * tid;
  int it = 0;
  for (int tile = first; tile < n_tiles; tile += stride, ++it) {
    const int buf = it & 1;
    const NfTileDesc& d = S.desc[it & 3];
    const bool have_next = tile + stride < n_tiles;
    int32_t dword = 0;                       // descriptor of tile it+3 (stored after the barrier)
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
    const uint32_t sAU = smem_u32(S.arena[buf]), sAD = sAU + 8u * (uint32_t)d.up.cn;
    uint16_t* sxD = S.sidx[buf][0];
    uint16_t* sxU = S.sidx[buf][1];
    // wait for the staged runs of this tile (each barrier serves every other tile)
    while (!mbar_try_wait(&S.full[buf], (uint32_t)((it >> 1) & 1))) {}
    // ---- phase 0 -------------------------------------------------------------------------------
    if (flag == NF_STAGED) {
      nf_slice_index(d.up, sAU, kc.uB.w, kc.uB.z, kc.uC.y, sxU, tid);
      nf_slice_index(d.dn, sAD, kc.dB.w, kc.dB.z, kc.dC.y, sxD, tid);
    }
    __syncthreads();          // slice index complete; every thread is done with the previous tile (other buffer free)
    if (tid == 0 && have_next) issue(S.desc[(it + 1) & 3], buf ^ 1);
    if (fetch3) reinterpret_cast<int32_t*>(&S.desc[(it + 3) & 3])[tid] = dword;
    // ---- phases A + B (thread = cluster) ---------------------------------------------------------
    if (tid < n) {
      int32_t bu = -1, bd = -1;
      float best = 0.0f;
      bool slow = false;
      if (flag == NF_STAGED) {
        // z slices the two windows touch (monotone key function: a superset of the window), as staged runs
        const int ud0 = bin_range(__fsub_rn(c.y, kc.uA.w), kc.uB.w, kc.uB.z, kc.uC.y) - d.up.s0;
        const int ud1 = bin_range(__fadd_rn(c.y, kc.uA.w), kc.uB.w, kc.uB.z, kc.uC.y) - d.up.s0;
        const int dd0 = bin_range(__fsub_rn(c.y, kc.dA.w), kc.dB.w, kc.dB.z, kc.dC.y) - d.dn.s0;
        const int dd1 = bin_range(__fadd_rn(c.y, kc.dA.w), kc.dB.w, kc.dB.z, kc.dC.y) - d.dn.s0;
        if (ud0 < 0 || ud1 >= d.up.nsl || dd0 < 0 || dd1 >= d.dn.nsl) {
          slow = true;                                  // not covered by the staged slices
        } else {
          const int ju0 = sxU[ud0], ju1 = sxU[ud1 + 1], jd0 = sxD[dd0], jd1 = sxD[dd1 + 1];
          const int nd = nf_test_run<K>(c, sAD, jd0, jd1, kc.dA.x, kc.dA.y, sListD);
          const int nu = nd > 0 ? nf_test_run<K>(c, sAU, ju0, ju1, kc.uA.x, kc.uA.y, sListU) : 0;
          if (nd > K || nu > K) {                       // dense region: no lists, nested loops over the runs
            int iu, id;
            if (nf_medium(c, sAU, ju0, ju1, sAD, jd0, jd1, kc.uA, kc.dA, g, best, iu, id)) {
              if (iu >= 0) { bu = iu + d.up.c0; bd = id + d.dn.c0; }
            } else {
              slow = true;
            }
          } else if (nu > 0) {
            // down vectors once: (y_c - y_d) * dxu = (y_d - y_c) * (-dxu), exact
#pragma unroll 1
            for (int k = 0; k < nd; ++k) {
              const float2 v = lds_f2(sAD + 8u * lds_u16(sListD + (uint32_t)k * kIdxRow));
              sts_f2(sVec + (uint32_t)k * kVecRow, __fmul_rn(__fsub_rn(v.x, c.x), -g.x), __fmul_rn(__fsub_rn(v.y, c.y), -g.x));
            }
            best = __int_as_float(0x7f800000);
            int bi = 0, bk = 0;
            bool tie = false;
#pragma unroll 1
            for (int i = 0; i < nu; ++i) {
              const uint32_t ju = lds_u16(sListU + (uint32_t)i * kIdxRow);
              const float2 v = lds_f2(sAU + 8u * ju);
              const float Ay = __fmul_rn(__fsub_rn(v.x, c.x), g.y), Az = __fmul_rn(__fsub_rn(v.y, c.y), g.y);
              uint32_t pb = sVec;
#pragma unroll 1
              for (int k = 0; k < nd; ++k, pb += kVecRow) {
                const float2 b = lds_f2(pb);
                const float ay = __fsub_rn(Ay, b.x), az = __fsub_rn(Az, b.y);
                const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
                tie = tie || (sc == best);
                if (sc < best) { best = sc; bi = (int)ju; bk = k; }
              }
            }
            if (tie) slow = true;
            else { bu = bi + d.up.c0; bd = (int32_t)lds_u16(sListD + (uint32_t)bk * kIdxRow) + d.dn.c0; }
          }
        }
      } else if (flag == NF_GLOBAL) {
        slow = true;
      }
      if (slow) {
        const int s = (d.rsf >> 8) & 0xff;
        nf_slow(c, kc, bin_start + (size_t)s * nbp1, syz + d.sec_off, order + d.sec_off, best, bu, bd);
      }
      if (!(bu >= 0 && best <= g.z)) { bu = -1; bd = -1; }
      link_up[d.p0 + tid] = bu;
      link_dn[d.p0 + tid] = bd;
    }
    // no barrier here: the next tile uses the other staging buffer and the other slice index; its phases A / B
    // write only the thread's own list / vector columns.
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
