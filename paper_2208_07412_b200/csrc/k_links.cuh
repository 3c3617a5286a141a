// S2 neighbour finder, S3 link cleaner, S4 start hits.
#pragma once
#include "k_grid.cuh"

namespace tpcca {

constexpr int kNfK = 6;        // window candidates cached per side and thread in shared memory
constexpr int kNfThreads = 256;

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

// Window candidates of one side (A, B, C = the side's NfConst groups): every cluster q of the
// neighbour row with |y_q - y_c| <= hy and |z_q - z_c| <= hz.  The bin range is a superset of the
// window; the z slices of the range are walked as ONE flattened loop so that the
// lanes of a warp, whose slices hold different numbers of clusters, stay together.
// Caches (dy * dxo, dz * dxo) and q of the first kNfK hits; returns the number of hits.
// UP: the cached vector is (y_q - y_c) * dxo; down side: (y_c - y_q) * dxo (fl(a - b) = -fl(b - a),
// so the negation is exact).
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

// Slow path of S2 for a cluster with more than kNfK window candidates on a side (dense noise):
// the full U x D product by nested rescans of both windows.
__device__ __noinline__ void nf_slow(const float2 c, const NfConst* __restrict__ kc, const uint32_t* __restrict__ bs,
                                     const float2* __restrict__ yz, const int32_t* __restrict__ ord,
                                     float& best, int32_t& bu, int32_t& bd) {
  const float4 dA = kc->dA, dB = kc->dB, uA = kc->uA, uB = kc->uB, g = kc->g;
  const int4 dC = kc->dC, uC = kc->uC;
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

// ---- K2: neighbour finder, one thread per cluster ------------------------
// For cluster c of row r (1 <= r <= n_rows-2): over U x D (exact windows in rows r+1, r-1) the
// pair minimising score = ay^2 + az^2, ay = (yu-yc)*dxd - (yc-yd)*dxu; ties -> smallest original
// id of u, then of d; stored if score <= nf_cut[r].
// A tile = kNfThreads consecutive sorted clusters of ONE row, so every per-row constant is block
// uniform (seven 128-bit loads); blocks walk the tile list with a grid stride.  Three flattened,
// warp-friendly loops per thread: gather D, gather U (window hits cached in shared memory), then
// the nu * nd pair scores.
__global__ void __launch_bounds__(kNfThreads)
k_neighbours(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
             const float2* __restrict__ syz, const uint32_t* __restrict__ bin_start,
             const int32_t* __restrict__ row_start, const int32_t* __restrict__ order,
             const int32_t* __restrict__ nf_tile_start, const int2* __restrict__ nf_desc,
             int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
  __shared__ float2 s_uv[kNfK][kNfThreads];
  __shared__ float2 s_dv[kNfK][kNfThreads];
  __shared__ int32_t s_ui[kNfK][kNfThreads];
  __shared__ int32_t s_di[kNfK][kNfThreads];
  const int n_rows = __ldg(&T->n_rows);
  const int n_tiles = __ldg(&nf_tile_start[__ldg(&T->n_sectors) * n_rows]);
  const size_t nbp1 = (size_t)__ldg(&T->bins_per_sector) + 1;
  const int tid = threadIdx.x;
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int2 td = __ldg(&nf_desc[tile]);
    const int s = td.x / n_rows, r = td.x - s * n_rows;
    const int32_t* rs = row_start + s * (n_rows + 1) + r;
    const int p = __ldg(&rs[0]) + td.y * kNfThreads + tid;
    if (p >= __ldg(&rs[1])) continue;
    const int off = __ldg(&sec[s].off);
    int32_t bu = -1, bd = -1;
    if (r >= 1 && r <= n_rows - 2) {
      const float2* yz = syz + off;
      const uint32_t* bs = bin_start + (size_t)s * nbp1;
      const NfConst* kc = &T->nf[r];
      const float2 c = yz[p];
      const float4 g = __ldg(&kc->g);
      const int nd = nf_gather<false>(c, __ldg(&kc->dA), __ldg(&kc->dB), __ldg(&kc->dC), g.x, bs, yz, s_dv, s_di, tid);
      const int nu = nf_gather<true>(c, __ldg(&kc->uA), __ldg(&kc->uB), __ldg(&kc->uC), g.y, bs, yz, s_uv, s_ui, tid);
      float best = 0.0f;
      if (nd <= kNfK && nu <= kNfK) {
        const int np = nu * nd;
        int iu = 0, id = 0, bi = -1, bj = 0;
        for (int k = 0; k < np; ++k) {
          const float2 a = s_uv[iu][tid], b = s_dv[id][tid];
          const float ay = __fsub_rn(a.x, b.x), az = __fsub_rn(a.y, b.y);
          const float sc = __fadd_rn(__fmul_rn(ay, ay), __fmul_rn(az, az));
          bool better = (bi < 0) || (sc < best);
          if (!better && sc == best) {
            const int32_t* ord = order + off;
            const int32_t u = s_ui[iu][tid], ub = s_ui[bi][tid];
            if (u != ub) better = __ldg(&ord[u]) < __ldg(&ord[ub]);
            else better = __ldg(&ord[s_di[id][tid]]) < __ldg(&ord[s_di[bj][tid]]);
          }
          if (better) { best = sc; bi = iu; bj = id; }
          if (++id == nd) { id = 0; ++iu; }
        }
        if (bi >= 0) { bu = s_ui[bi][tid]; bd = s_di[bj][tid]; }
      } else {
        nf_slow(c, kc, bs, yz, order + off, best, bu, bd);
      }
      if (!(bu >= 0 && best <= g.z)) { bu = -1; bd = -1; }
    }
    link_up[off + p] = bu;
    link_dn[off + p] = bd;
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
