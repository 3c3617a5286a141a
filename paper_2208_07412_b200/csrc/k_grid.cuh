// S1 grid build: counting sort of the clusters of every sector by
// (row, bin, original index).  histogram -> per-sector exclusive scan -> scatter -> in-bin fix-up.
#pragma once
#include "tpcca_dev.cuh"

namespace tpcca {

// S1 is a two-level sort.  Level 1 partitions the clusters of a sector into coarse
// buckets (row, z slab of kSlab slices) with a counting sort on L2-resident counters; level 2 sorts
// every bucket by (bin, original id) in shared memory and writes the sorted clusters and the
// bucket's bin_start entries with coalesced stores.  Nothing touches the 1.5 GB bin_start array
// with atomics and no pass runs over it except the one that writes it.
// z slices per coarse bucket = 1 << DevTables::slab_shift, chosen per context (slab_shift_for in tpcca_api.cu)
// so that a bucket holds a few hundred clusters at the context's capacity
constexpr int kSlabShiftMin = 5, kSlabShiftMax = 7;
#ifndef TPCCA_SORT_CAPR
#define TPCCA_SORT_CAPR 1536
#endif
constexpr int kSortCapR = TPCCA_SORT_CAPR;               // clusters of a bucket sorted in shared memory
constexpr int kSortCapB = 2048;               // fine bins of a bucket (slab * ny) handled in shared memory

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

// ---- zero n 32-bit words (grid-stride) ---------------------------------------------------------------
__global__ void __launch_bounds__(256) k_zero_words(uint32_t* __restrict__ p, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = 0u;
}

struct GridRec { float y, z; int32_t id; int32_t pad; };   // level-1 record (16 bytes, one 128-bit store)

// ---- K1a: level-1 histogram: cb_cnt[s][cb(row, bz >> kSlabShift)]++ ---------------------------------
__global__ void __launch_bounds__(256)
k_cb_count(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, uint32_t* __restrict__ cb_cnt,
           uint32_t* __restrict__ rank, DevStatus* __restrict__ st) {
  // consecutive blocks work on different sectors: the atomics of the blocks in flight are spread over the
  // counters of all sectors (36 x 58 KB) instead of hammering the few hundred cache lines of one
  const int ns = __ldg(&T->n_sectors);
  const int s = blockIdx.x % ns;
  const SectorDesc sd = sec[s];
  const int i = (blockIdx.x / ns) * 256 + threadIdx.x;
  if (i >= sd.n) return;
  const int r = sd.row[i];
  if (r >= __ldg(&T->n_rows)) { st->err_range = 1; return; }
  const int bz = bin_coord(sd.z[i], __ldg(&T->grid_z_lo), __ldg(&T->inv_bz[r]), __ldg(&T->nz_hi[r]));
  const int cb = __ldg(&T->cb_base[r]) + (bz >> __ldg(&T->slab_shift));
  // the arrival rank inside the bucket is kept: the scatter pass needs no second atomic
  rank[(size_t)sd.off + i] = atomicAdd(&cb_cnt[(size_t)s * (__ldg(&T->n_cb) + 1) + cb], 1u);
}

// ---- K1b: one block per sector: cb_start = exclusive scan of cb_cnt (sector-local) -----------------
__global__ void __launch_bounds__(1024)
k_cb_scan(const DevTables* __restrict__ T, const uint32_t* __restrict__ cb_cnt, uint32_t* __restrict__ cb_start) {
  __shared__ uint32_t ws[33];
  const int ncb = T->n_cb;
  const size_t base = (size_t)blockIdx.x * (ncb + 1);
  uint32_t carry = 0;
  for (int b0 = 0; b0 < ncb; b0 += 1024) {
    const int b = b0 + threadIdx.x;
    const uint32_t v = b < ncb ? cb_cnt[base + b] : 0u;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan<uint32_t>(v, ws, total);
    if (b < ncb) cb_start[base + b] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0) cb_start[base + ncb] = carry;
}

// ---- K1c: level-1 scatter: record (y, z, id) to slot cb_start + arrival rank of its bucket ----------
__global__ void __launch_bounds__(256)
k_cb_scatter(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, const uint32_t* __restrict__ cb_start,
             const uint32_t* __restrict__ rank, GridRec* __restrict__ rec) {
  const int ns = __ldg(&T->n_sectors);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].tile256); });
  const SectorDesc sd = sec[s];
  const int i = (blockIdx.x - sd.tile256) * 256 + threadIdx.x;
  if (i >= sd.n) return;
  const int r = sd.row[i];
  if (r >= __ldg(&T->n_rows)) return;
  const float y = sd.y[i], z = sd.z[i];
  const int bz = bin_coord(z, __ldg(&T->grid_z_lo), __ldg(&T->inv_bz[r]), __ldg(&T->nz_hi[r]));
  const int cb = __ldg(&T->cb_base[r]) + (bz >> __ldg(&T->slab_shift));
  const uint32_t pos = __ldg(&cb_start[(size_t)s * (__ldg(&T->n_cb) + 1) + cb]) + rank[(size_t)sd.off + i];
  GridRec o; o.y = y; o.z = z; o.id = i; o.pad = 0;
  *reinterpret_cast<float4*>(&rec[(size_t)sd.off + pos]) = *reinterpret_cast<const float4*>(&o);
}

// row and slab of a coarse bucket: largest r with cb_base[r] <= cb
__device__ __forceinline__ void cb_row_slab(const DevTables* __restrict__ T, int cb, int& r, int& k) {
  int lo = 0, hi = __ldg(&T->n_rows) - 1;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (__ldg(&T->cb_base[mid]) <= cb) lo = mid; else hi = mid - 1;
  }
  r = lo; k = cb - __ldg(&T->cb_base[lo]);
}

// ---- K1d: level 2, one block per (sector, coarse bucket) ------------------------------------------
// Counting sort of the bucket's clusters by fine bin in shared memory (arrival rank from the
// shared-memory histogram), then the canonical in-bin order (ascending original id) by counting the
// smaller ids of the same bin; writes syz / order (sorted positions) and the bucket's bin_start
// entries.  Buckets that do not fit the shared-memory buffers go to the big-bucket list.
__global__ void __launch_bounds__(256)
k_grid_sort(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, const int32_t* __restrict__ cb_rs,
            const uint32_t* __restrict__ cb_start,
            const GridRec* __restrict__ rec, float2* __restrict__ syz, int32_t* __restrict__ order,
            uint32_t* __restrict__ bin_start, uint32_t* __restrict__ big_list, DevStatus* __restrict__ st) {
  __shared__ float s_y[kSortCapR], s_z[kSortCapR];
  __shared__ int32_t s_id[kSortCapR];
  __shared__ uint16_t s_lb[kSortCapR], s_rank[kSortCapR], s_perm[kSortCapR];
  __shared__ uint32_t s_hist[kSortCapB + 8];
  __shared__ uint32_t ws[33];
  const int ncb = __ldg(&T->n_cb);
  const int s = blockIdx.x / ncb, cb = blockIdx.x - s * ncb;
  const int rs = __ldg(&cb_rs[cb]);             // host table: row | slab << 8 (no search per block)
  const int r = rs & 0xff, k = rs >> 8;
  const int ny = __ldg(&T->ny[r]), nz = __ldg(&T->nz[r]);
  const int kSlab = 1 << __ldg(&T->slab_shift);
  const int nsl = min(kSlab, nz - k * kSlab);
  const int nbins = nsl * ny;
  const uint32_t* cs = cb_start + (size_t)s * (ncb + 1) + cb;
  const uint32_t bstart = __ldg(&cs[0]);
  const int nb_ = (int)(__ldg(&cs[1]) - bstart);
  if (nb_ > kSortCapR || nbins > kSortCapB) {
    if (threadIdx.x == 0) big_list[atomicAdd(&st->n_big, 1u)] = blockIdx.x;
    return;
  }
  const int off = __ldg(&sec[s].off);
  const size_t gb0 = (size_t)s * (__ldg(&T->bins_per_sector) + 1) + __ldg(&T->bin_base[r]) + (size_t)k * kSlab * ny;
  for (int j = threadIdx.x; j < nbins; j += 256) s_hist[j] = 0;
  __syncthreads();
  const float ylo = __ldg(&T->y_lo[r]), iby = __ldg(&T->inv_by[r]), nyh = __ldg(&T->ny_hi[r]);
  const float zlo = __ldg(&T->grid_z_lo), ibz = __ldg(&T->inv_bz[r]), nzh = __ldg(&T->nz_hi[r]);
  for (int i = threadIdx.x; i < nb_; i += 256) {
    const float4 q = __ldg(reinterpret_cast<const float4*>(&rec[(size_t)off + bstart + i]));
    const int by = bin_coord(q.x, ylo, iby, nyh), bz = bin_coord(q.y, zlo, ibz, nzh);
    const int lb = (bz - k * kSlab) * ny + by;
    s_y[i] = q.x; s_z[i] = q.y; s_id[i] = __float_as_int(q.z);
    s_lb[i] = (uint16_t)lb;
    s_rank[i] = (uint16_t)atomicAdd(&s_hist[lb], 1u);
  }
  __syncthreads();
  // exclusive scan of the bin counts (8 consecutive bins per thread), in place; s_hist[nbins] = nb_
  {
    const int b0 = threadIdx.x * 8;
    uint32_t cnt[8], v = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { cnt[j] = (b0 + j < nbins) ? s_hist[b0 + j] : 0u; v += cnt[j]; }
    uint32_t total;
    uint32_t run = block_exclusive_scan<uint32_t>(v, ws, total);
#pragma unroll
    for (int j = 0; j < 8; ++j) { if (b0 + j < nbins) s_hist[b0 + j] = run; run += cnt[j]; }
    if (threadIdx.x == 0) s_hist[nbins] = (uint32_t)nb_;
  }
  __syncthreads();
  // bin_start of the bucket's bins; entry nbins (= first bin of the next bucket, or the sector's
  // closing entry) is written with the same value by its own bucket as well
  for (int j = threadIdx.x; j <= nbins; j += 256) bin_start[gb0 + j] = bstart + s_hist[j];
  for (int i = threadIdx.x; i < nb_; i += 256) s_perm[s_hist[s_lb[i]] + s_rank[i]] = (uint16_t)i;
  __syncthreads();
  for (int i = threadIdx.x; i < nb_; i += 256) {
    const int lb = s_lb[i];
    const uint32_t lo = s_hist[lb], hi = s_hist[lb + 1];
    uint32_t pos = lo;
    if (hi - lo > 1) {
      const int32_t id = s_id[i];
      for (uint32_t q = lo; q < hi; ++q) pos += (s_id[s_perm[q]] < id) ? 1u : 0u;
    }
    const size_t g = (size_t)off + bstart + pos;
    syz[g] = make_float2(s_y[i], s_z[i]);
    order[g] = s_id[i];
  }
}

// ---- K1e: buckets too large for shared memory: one block per listed bucket, global memory -----------
// counts in bin_start[gb0 + 1 + lb], exclusive scan in place (entry j + 1 = start of bin j), scatter
// with the cursor trick (afterwards entry j + 1 = end of bin j = start of bin j + 1), then insertion
// sort by original id inside every bin with more than one cluster.
__global__ void __launch_bounds__(256)
k_grid_big(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec, const uint32_t* __restrict__ cb_start,
           const GridRec* __restrict__ rec, float2* __restrict__ syz, int32_t* __restrict__ order,
           uint32_t* __restrict__ bin_start, const uint32_t* __restrict__ big_list, const DevStatus* __restrict__ st) {
  __shared__ uint32_t ws[33];
  __shared__ uint32_t s_carry;
  const int ncb = __ldg(&T->n_cb);
  const uint32_t n_big = st->n_big;
  for (uint32_t bi = blockIdx.x; bi < n_big; bi += gridDim.x) {
    const int bid = (int)big_list[bi];
    const int s = bid / ncb, cb = bid - s * ncb;
    int r, k;
    cb_row_slab(T, cb, r, k);
    const int ny = __ldg(&T->ny[r]), nz = __ldg(&T->nz[r]);
    const int kSlab = 1 << __ldg(&T->slab_shift);
    const int nsl = min(kSlab, nz - k * kSlab);
    const int nbins = nsl * ny;
    const uint32_t* cs = cb_start + (size_t)s * (ncb + 1) + cb;
    const uint32_t bstart = cs[0];
    const int nb_ = (int)(cs[1] - bstart);
    const int off = sec[s].off;
    uint32_t* bs = bin_start + (size_t)s * (__ldg(&T->bins_per_sector) + 1) + __ldg(&T->bin_base[r]) + (size_t)k * kSlab * ny;
    const float ylo = __ldg(&T->y_lo[r]), iby = __ldg(&T->inv_by[r]), nyh = __ldg(&T->ny_hi[r]);
    const float zlo = __ldg(&T->grid_z_lo), ibz = __ldg(&T->inv_bz[r]), nzh = __ldg(&T->nz_hi[r]);
    auto local_bin = [&](float y, float z) {
      return (bin_coord(z, zlo, ibz, nzh) - k * kSlab) * ny + bin_coord(y, ylo, iby, nyh);
    };
    for (int j = 1 + threadIdx.x; j <= nbins; j += 256) bs[j] = 0;    // entry 0 belongs to the previous bucket
    __syncthreads();
    for (int i = threadIdx.x; i < nb_; i += 256) {
      const GridRec q = rec[(size_t)off + bstart + i];
      atomicAdd(&bs[1 + local_bin(q.y, q.z)], 1u);
    }
    if (threadIdx.x == 0) s_carry = bstart;
    __syncthreads();
    for (int b0 = 0; b0 < nbins; b0 += 256) {      // bs[1 + j] = bstart + (clusters in bins < j)
      const int j = b0 + threadIdx.x;
      const uint32_t v = j < nbins ? bs[1 + j] : 0u;
      uint32_t total;
      const uint32_t ex = block_exclusive_scan<uint32_t>(v, ws, total);
      const uint32_t carry = s_carry;
      if (j < nbins) bs[1 + j] = carry + ex;
      __syncthreads();
      if (threadIdx.x == 0) s_carry = carry + total;
      __syncthreads();
    }
    if (threadIdx.x == 0 && cb == 0) bs[0] = bstart;
    __syncthreads();
    for (int i = threadIdx.x; i < nb_; i += 256) {
      const GridRec q = rec[(size_t)off + bstart + i];
      const uint32_t pos = atomicAdd(&bs[1 + local_bin(q.y, q.z)], 1u);
      syz[(size_t)off + pos] = make_float2(q.y, q.z);
      order[(size_t)off + pos] = q.id;
    }
    __syncthreads();
    for (int j = threadIdx.x; j < nbins; j += 256) {
      const uint32_t lo = j == 0 ? bstart : bs[j], hi = bs[j + 1];
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
    __syncthreads();
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
             int32_t* __restrict__ row_start, int32_t* __restrict__ nf_tile_start, const DevStatus* __restrict__ st) {
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
      v = st->err_range ? 0 : (cnt + kNfTile - 1) / kNfTile;     // a failed S1 (TPCCA_E_RANGE) leaves S2 nothing to do
    }
    int total;
    const int ex = block_exclusive_scan<int>(v, ws, total);
    if (i < n) nf_tile_start[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0) nf_tile_start[n] = carry;
}

}  // namespace tpcca
