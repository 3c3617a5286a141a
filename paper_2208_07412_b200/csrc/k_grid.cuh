// S1 grid build: counting sort of the clusters of every sector by
// (row, bin, original index).  histogram -> per-sector exclusive scan -> scatter -> in-bin fix-up.
#pragma once
#include "tpcca_dev.cuh"

namespace tpcca {

constexpr int kScanTile = 2048;     // bins per scan tile (256 threads x 8)

// sector of a tile: largest s with first_tile(s) <= tile (sectors with no tiles are skipped
// because their first tile equals the next sector's).
template <class F>
__device__ __forceinline__ int find_sector(int ns, int tile, F first_tile) {
  int lo = 0, hi = ns - 1;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (first_tile(mid) <= tile) lo = mid; else hi = mid - 1;
  }
  return lo;
}

__device__ __forceinline__ int cluster_key(const DevTables* __restrict__ T, int r, float y, float z) {
  int by = bin_coord(y, __ldg(&T->y_lo[r]), __ldg(&T->inv_by[r]), __ldg(&T->ny_hi[r]));
  int bz = bin_coord(z, __ldg(&T->grid_z_lo), __ldg(&T->inv_bz[r]), __ldg(&T->nz_hi[r]));
  return __ldg(&T->bin_base[r]) + bz * __ldg(&T->ny[r]) + by;
}

// ---- K1a: histogram.  cnt = bin_start + 1 (the cursor trick of DESIGN.md 5.1): cnt[s][key]++.
// The thread that makes a bin's count 2 records the bin in the multi-bin list.
__global__ void __launch_bounds__(256)
k_grid_count(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
             uint32_t* __restrict__ bin_start, uint32_t* __restrict__ multi_list, uint32_t multi_cap,
             DevStatus* __restrict__ st) {
  const int ns = __ldg(&T->n_sectors);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].tile256); });
  const SectorDesc sd = sec[s];
  const int i = (blockIdx.x - sd.tile256) * 256 + threadIdx.x;
  bool is_multi = false;
  uint32_t slot = 0;
  if (i < sd.n) {
    const int r = sd.row[i];
    if (r >= __ldg(&T->n_rows)) {
      st->err_range = 1;
    } else {
      const int key = cluster_key(T, r, sd.y[i], sd.z[i]);
      slot = (uint32_t)s * (uint32_t)(__ldg(&T->bins_per_sector) + 1) + 1u + (uint32_t)key;
      const uint32_t old = atomicAdd(&bin_start[slot], 1u);
      is_multi = (old == 1u);
    }
  }
  // warp-aggregated append to the multi-bin list
  const unsigned m = __ballot_sync(0xffffffffu, is_multi);
  if (m) {
    const int lane = threadIdx.x & 31;
    uint32_t base = 0;
    if (lane == (__ffs(m) - 1)) base = atomicAdd(&st->n_multi, (uint32_t)__popc(m));
    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
    if (is_multi) {
      const uint32_t k = base + (uint32_t)__popc(m & ((1u << lane) - 1u));
      if (k < multi_cap) multi_list[k] = slot;
    }
  }
}

// ---- K1b: per-tile sums of the bin counts (tiles never cross a sector) ------------------------
__global__ void __launch_bounds__(256)
k_scan_tile_sums(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
                 const uint32_t* __restrict__ bin_start, uint32_t* __restrict__ tile_sum) {
  __shared__ uint32_t ws[33];
  const int ns = __ldg(&T->n_sectors);
  const int nb = __ldg(&T->bins_per_sector);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].bin_tile); });
  const int t = blockIdx.x - __ldg(&sec[s].bin_tile);
  const uint32_t* a = bin_start + (size_t)s * (nb + 1) + 1;   // cnt[0..nb)
  const int b0 = t * kScanTile + threadIdx.x * 8;
  uint32_t v = 0;
  if (b0 + 8 <= nb && ((((size_t)s * (nb + 1) + 1 + b0) & 3) == 0)) {
    const uint4 q0 = *reinterpret_cast<const uint4*>(a + b0);
    const uint4 q1 = *reinterpret_cast<const uint4*>(a + b0 + 4);
    v = q0.x + q0.y + q0.z + q0.w + q1.x + q1.y + q1.z + q1.w;
  } else {
    for (int k = 0; k < 8; ++k) if (b0 + k < nb) v += a[b0 + k];
  }
  uint32_t total;
  block_exclusive_scan<uint32_t>(v, ws, total);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

// ---- K1c: one block per sector scans that sector's tile sums (exclusive, in place) ------------
__global__ void __launch_bounds__(1024)
k_scan_sector_tiles(const SectorDesc* __restrict__ sec, uint32_t* __restrict__ tile_sum) {
  __shared__ uint32_t ws[33];
  const int s = blockIdx.x;
  const int t0 = sec[s].bin_tile, t1 = sec[s + 1].bin_tile;
  uint32_t carry = 0;
  for (int base = t0; base < t1; base += 1024) {
    const int t = base + threadIdx.x;
    const uint32_t v = t < t1 ? tile_sum[t] : 0u;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan<uint32_t>(v, ws, total);
    if (t < t1) tile_sum[t] = carry + ex;
    carry += total;
  }
}

// ---- K1d: apply: bin_start[s][1 + b] = exclusive prefix of the counts (sector-local) ----------
__global__ void __launch_bounds__(256)
k_scan_apply(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
             uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ tile_sum) {
  __shared__ uint32_t ws[33];
  const int ns = __ldg(&T->n_sectors);
  const int nb = __ldg(&T->bins_per_sector);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].bin_tile); });
  const int t = blockIdx.x - __ldg(&sec[s].bin_tile);
  uint32_t* a = bin_start + (size_t)s * (nb + 1) + 1;
  const int b0 = t * kScanTile + threadIdx.x * 8;
  uint32_t c[8];
  uint32_t v = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) { c[k] = (b0 + k < nb) ? a[b0 + k] : 0u; v += c[k]; }
  uint32_t total;
  uint32_t run = block_exclusive_scan<uint32_t>(v, ws, total) + tile_sum[blockIdx.x];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    if (b0 + k < nb) a[b0 + k] = run;
    run += c[k];
  }
}

// ---- K1e: scatter.  pos = cursor[key]++ (arrival order inside a bin; K1f restores id order).
// Afterwards bin_start[s][j] = first position of bin j for every j in [0, nb] (cursor trick).
__global__ void __launch_bounds__(256)
k_grid_scatter(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
               uint32_t* __restrict__ bin_start, float2* __restrict__ syz, int32_t* __restrict__ order) {
  const int ns = __ldg(&T->n_sectors);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].tile256); });
  const SectorDesc sd = sec[s];
  const int i = (blockIdx.x - sd.tile256) * 256 + threadIdx.x;
  if (i >= sd.n) return;
  const int r = sd.row[i];
  if (r >= __ldg(&T->n_rows)) return;
  const float y = sd.y[i], z = sd.z[i];
  const int key = cluster_key(T, r, y, z);
  uint32_t* cur = bin_start + (size_t)s * (__ldg(&T->bins_per_sector) + 1) + 1;
  const uint32_t pos = atomicAdd(&cur[key], 1u);
  const size_t g = (size_t)sd.off + pos;
  syz[g] = make_float2(y, z);
  order[g] = i;
}

// ---- K1f: bins with >= 2 clusters: insertion sort by original index (canonical order) --------
__global__ void __launch_bounds__(256)
k_grid_fixup(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
             const uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ multi_list,
             const DevStatus* __restrict__ st, float2* __restrict__ syz, int32_t* __restrict__ order) {
  const uint32_t n_multi = st->n_multi;
  const uint32_t stride = (uint32_t)(__ldg(&T->bins_per_sector) + 1);
  for (uint32_t k = blockIdx.x * blockDim.x + threadIdx.x; k < n_multi; k += gridDim.x * blockDim.x) {
    const uint32_t slot = multi_list[k];         // = s*stride + 1 + key
    const uint32_t s = slot / stride;
    const size_t off = (size_t)sec[s].off;
    const uint32_t lo = bin_start[slot - 1], hi = bin_start[slot];
    for (uint32_t a = lo + 1; a < hi; ++a) {
      const int32_t oa = order[off + a];
      const float2 va = syz[off + a];
      uint32_t b = a;
      while (b > lo && order[off + b - 1] > oa) {
        order[off + b] = order[off + b - 1];
        syz[off + b] = syz[off + b - 1];
        --b;
      }
      order[off + b] = oa;
      syz[off + b] = va;
    }
  }
}

// ---- K1g: row_start[s][r] = bin_start[s][bin_base[r]], and the row-aligned tiling of S2 ---------
// One block.  nf_tile_start[i], i = s * n_rows + r: first S2 tile of (sector s, row r); a tile is
// kNfTile consecutive sorted clusters of ONE row; nf_tile_start[ns * n_rows] = total.
#ifndef TPCCA_NF_TILE
#define TPCCA_NF_TILE 128
#endif
constexpr int kNfTile = TPCCA_NF_TILE;

__global__ void __launch_bounds__(1024)
k_row_tables(const DevTables* __restrict__ T, const uint32_t* __restrict__ bin_start,
             int32_t* __restrict__ row_start, int32_t* __restrict__ nf_tile_start) {
  __shared__ int ws[33];
  const int nr = T->n_rows, ns = T->n_sectors;
  const size_t stride = (size_t)T->bins_per_sector + 1;
  for (int i = threadIdx.x; i < ns * (nr + 1); i += blockDim.x) {
    const int s = i / (nr + 1), r = i - s * (nr + 1);
    row_start[i] = (int32_t)bin_start[s * stride + T->bin_base[r]];
  }
  __syncthreads();
  int carry = 0;
  const int n = ns * nr;
  for (int base = 0; base < n; base += 1024) {
    const int i = base + threadIdx.x;
    int v = 0;
    if (i < n) {
      const int s = i / nr, r = i - s * nr;
      const int cnt = row_start[s * (nr + 1) + r + 1] - row_start[s * (nr + 1) + r];
      v = (cnt + kNfTile - 1) / kNfTile;
    }
    int total;
    const int ex = block_exclusive_scan<int>(v, ws, total);
    if (i < n) nf_tile_start[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0) nf_tile_start[n] = carry;
}

}  // namespace tpcca
