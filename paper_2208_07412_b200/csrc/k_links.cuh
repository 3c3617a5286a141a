// S2 neighbour finder, S3 link cleaner, S4 start hits.
#pragma once
#include "k_grid.cuh"

namespace tpcca {

constexpr int kNfKD = 8;   // down-candidates cached per thread in shared memory

// row of sorted position p: rows are contiguous runs; start from the block's first row.
__device__ __forceinline__ int row_of(const int32_t* __restrict__ rs, int r, int p) {
  while (p >= __ldg(&rs[r + 1])) ++r;
  return r;
}
__device__ __forceinline__ int row_search(const int32_t* __restrict__ rs, int n_rows, int p) {
  int lo = 0, hi = n_rows - 1;               // largest r with rs[r] <= p
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (__ldg(&rs[mid]) <= p) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// ---- K2: neighbour finder, one thread per cluster -----------------------------
// For cluster c of row r (1 <= r <= n_rows-2): over U x D (exact windows in rows r+1, r-1) the
// pair minimising score = ay^2 + az^2, ay = (yu-yc)*dxd - (yc-yd)*dxu; ties -> smallest original
// id of u, then of d; stored if score <= nf_cut[r].
__global__ void __launch_bounds__(256)
k_neighbours(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
             const float2* __restrict__ syz, const uint32_t* __restrict__ bin_start,
             const int32_t* __restrict__ row_start, const int32_t* __restrict__ order,
             int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  __shared__ float s_by[kNfKD][256];
  __shared__ float s_bz[kNfKD][256];
  __shared__ int32_t s_id[kNfKD][256];
  __shared__ int s_r0;
  const int ns = __ldg(&T->n_sectors);
  const int n_rows = __ldg(&T->n_rows);
  const int s = find_sector(ns, blockIdx.x, [&](int i) { return __ldg(&sec[i].tile256); });
  const int n = __ldg(&sec[s].n), off = __ldg(&sec[s].off);
  const int p0 = (blockIdx.x - __ldg(&sec[s].tile256)) * 256;
  const int32_t* rs = row_start + s * (n_rows + 1);
  if (threadIdx.x == 0) s_r0 = row_search(rs, n_rows, p0);
  __syncthreads();
  const int p = p0 + threadIdx.x;
  if (p >= n) return;
  const int tid = threadIdx.x;
  const int r = row_of(rs, s_r0, p);
  const float2* yz = syz + off;
  const int32_t* ord = order + off;
  const uint32_t* bs = bin_start + (size_t)s * (__ldg(&T->bins_per_sector) + 1);
  int32_t bu = -1, bd = -1;
  if (r >= 1 && r <= n_rows - 2) {
    const float2 c = yz[p];
    const float margin = __ldg(&T->margin);
    const float dxu = __fsub_rn(__ldg(&T->row_x[r + 1]), __ldg(&T->row_x[r]));
    const float dxd = __fsub_rn(__ldg(&T->row_x[r]), __ldg(&T->row_x[r - 1]));
    // ---- pass 1: down window (row r-1): cache (By, Bz, id)
    int nd = 0;
    {
      const int r2 = r - 1;
      const float hy = __ldg(&T->hy_dn[r]), hz = __ldg(&T->hz_dn[r]);
      const float my = __fadd_rn(hy, margin), mz = __fadd_rn(hz, margin);
      const float ylo = __ldg(&T->y_lo[r2]), iby = __ldg(&T->inv_by[r2]), nyh = __ldg(&T->ny_hi[r2]);
      const float zlo = __ldg(&T->grid_z_lo), ibz = __ldg(&T->inv_bz[r2]), nzh = __ldg(&T->nz_hi[r2]);
      const int by0 = bin_coord(__fsub_rn(c.x, my), ylo, iby, nyh), by1 = bin_coord(__fadd_rn(c.x, my), ylo, iby, nyh);
      const int bz0 = bin_coord(__fsub_rn(c.y, mz), zlo, ibz, nzh), bz1 = bin_coord(__fadd_rn(c.y, mz), zlo, ibz, nzh);
      const int ny = __ldg(&T->ny[r2]);
      const int base = __ldg(&T->bin_base[r2]);
      for (int bz = bz0; bz <= bz1; ++bz) {
        const int b0 = base + bz * ny;
        const uint32_t e = __ldg(&bs[b0 + by1 + 1]);
        for (uint32_t q = __ldg(&bs[b0 + by0]); q < e; ++q) {
          const float2 d = __ldg(&yz[q]);
          const float dy = __fsub_rn(d.x, c.x), dz = __fsub_rn(d.y, c.y);
          if (fabsf(dy) <= hy && fabsf(dz) <= hz) {
            if (nd < kNfKD) {
              s_by[nd][tid] = __fmul_rn(__fsub_rn(c.x, d.x), dxu);
              s_bz[nd][tid] = __fmul_rn(__fsub_rn(c.y, d.y), dxu);
              s_id[nd][tid] = (int32_t)q;
            }
            ++nd;
          }
        }
      }
    }
    if (nd > 0) {
      // ---- pass 2: up window (row r+1); score against the cached (or re-scanned) D
      const int r2 = r + 1;
      const float hy = __ldg(&T->hy_up[r]), hz = __ldg(&T->hz_up[r]);
      const float my = __fadd_rn(hy, margin), mz = __fadd_rn(hz, margin);
      const float ylo = __ldg(&T->y_lo[r2]), iby = __ldg(&T->inv_by[r2]), nyh = __ldg(&T->ny_hi[r2]);
      const float zlo = __ldg(&T->grid_z_lo), ibz = __ldg(&T->inv_bz[r2]), nzh = __ldg(&T->nz_hi[r2]);
      const int by0 = bin_coord(__fsub_rn(c.x, my), ylo, iby, nyh), by1 = bin_coord(__fadd_rn(c.x, my), ylo, iby, nyh);
      const int bz0 = bin_coord(__fsub_rn(c.y, mz), zlo, ibz, nzh), bz1 = bin_coord(__fadd_rn(c.y, mz), zlo, ibz, nzh);
      const int ny = __ldg(&T->ny[r2]);
      const int base = __ldg(&T->bin_base[r2]);
      float best = 0.0f;
      bool have = false;
      auto consider = [&](float s, int32_t u, int32_t d) {
        bool better;
        if (!have) better = true;
        else if (s < best) better = true;
        else if (s == best) {
          const int32_t ou = __ldg(&ord[u]), obu = __ldg(&ord[bu]);
          if (ou != obu) better = ou < obu;
          else better = __ldg(&ord[d]) < __ldg(&ord[bd]);
        } else better = false;
        if (better) { have = true; best = s; bu = u; bd = d; }
      };
      for (int bz = bz0; bz <= bz1; ++bz) {
        const int b0 = base + bz * ny;
        const uint32_t e = __ldg(&bs[b0 + by1 + 1]);
        for (uint32_t q = __ldg(&bs[b0 + by0]); q < e; ++q) {
          const float2 u = __ldg(&yz[q]);
          const float dy = __fsub_rn(u.x, c.x), dz = __fsub_rn(u.y, c.y);
          if (!(fabsf(dy) <= hy && fabsf(dz) <= hz)) continue;
          const float Ay = __fmul_rn(dy, dxd), Az = __fmul_rn(dz, dxd);
          if (nd <= kNfKD) {
            for (int k = 0; k < nd; ++k) {
              const float ay = __fsub_rn(Ay, s_by[k][tid]);
              const float az = __fsub_rn(Az, s_bz[k][tid]);
              const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
              consider(sc, (int32_t)q, s_id[k][tid]);
            }
          } else {
            // overflow (dense noise): re-scan the down window for this u
            const int rd = r - 1;
            const float hyd = __ldg(&T->hy_dn[r]), hzd = __ldg(&T->hz_dn[r]);
            const float myd = __fadd_rn(hyd, margin), mzd = __fadd_rn(hzd, margin);
            const float ylod = __ldg(&T->y_lo[rd]), ibyd = __ldg(&T->inv_by[rd]), nyhd = __ldg(&T->ny_hi[rd]);
            const float ibzd = __ldg(&T->inv_bz[rd]), nzhd = __ldg(&T->nz_hi[rd]);
            const int dy0 = bin_coord(__fsub_rn(c.x, myd), ylod, ibyd, nyhd), dy1 = bin_coord(__fadd_rn(c.x, myd), ylod, ibyd, nyhd);
            const int dz0 = bin_coord(__fsub_rn(c.y, mzd), zlo, ibzd, nzhd), dz1 = bin_coord(__fadd_rn(c.y, mzd), zlo, ibzd, nzhd);
            const int nyd = __ldg(&T->ny[rd]);
            const int based = __ldg(&T->bin_base[rd]);
            for (int bzd = dz0; bzd <= dz1; ++bzd) {
              const int bd0 = based + bzd * nyd;
              const uint32_t ed = __ldg(&bs[bd0 + dy1 + 1]);
              for (uint32_t qd = __ldg(&bs[bd0 + dy0]); qd < ed; ++qd) {
                const float2 d = __ldg(&yz[qd]);
                const float ddy = __fsub_rn(d.x, c.x), ddz = __fsub_rn(d.y, c.y);
                if (!(fabsf(ddy) <= hyd && fabsf(ddz) <= hzd)) continue;
                const float ay = __fsub_rn(Ay, __fmul_rn(__fsub_rn(c.x, d.x), dxu));
                const float az = __fsub_rn(Az, __fmul_rn(__fsub_rn(c.y, d.y), dxu));
                const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
                consider(sc, (int32_t)q, (int32_t)qd);
              }
            }
          }
        }
      }
      if (!(have && best <= __ldg(&T->nf_cut[r]))) { bu = -1; bd = -1; }
    }
  }
  link_up[off + p] = bu;
  link_dn[off + p] = bd;
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
