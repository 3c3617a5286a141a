// Device-side data structures shared by the tpcca kernels (product code; no oracle code here).
// Layout in HBM: DESIGN.md section 4.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/tpcca.h"

namespace tpcca {

constexpr int kMaxRows = TPCCA_MAX_ROWS;
constexpr int kMaxSectors = TPCCA_MAX_SECTORS;

// Per-row tables, copied verbatim from tpcca_params (DESIGN.md 3 "Derived tables").  Lives in
// global memory; kernels read it through the read-only path (uniform per warp in S1-S4) or stage
// the rows they need in shared memory (S5, where lanes sit on different rows).
// S2 constants of one row r (1 <= r <= n_rows-2), 16-byte groups so that a thread fetches them
// with seven 128-bit loads (block-uniform address).  d* = towards row r-1, u* = towards row r+1.
struct NfConst {
  float4 dA;   // hy_dn, hz_dn, hy_dn + margin, hz_dn + margin
  float4 dB;   // y_lo[r-1], inv_by[r-1], inv_bz[r-1], grid_z_lo
  int4 dC;     // ny[r-1] - 1, nz[r-1] - 1, ny[r-1], bin_base[r-1]
  float4 uA;   // hy_up, hz_up, hy_up + margin, hz_up + margin
  float4 uB;   // y_lo[r+1], inv_by[r+1], inv_bz[r+1], grid_z_lo
  int4 uC;     // ny[r+1] - 1, nz[r+1] - 1, ny[r+1], bin_base[r+1]
  float4 g;    // dxu = x[r+1] - x[r], dxd = x[r] - x[r-1], nf_cut[r], 0
};

struct DevTables {
  int32_t n_rows, n_sectors;
  int32_t bins_per_sector;              // nb = sum_r ny_r * nz_r
  int32_t tc_max_gap, tc_min_hits;
  int32_t sel_permille;                 // S6: max shared hits of a selected tracklet, in 1/1000 of its hits
  float res_inv_q;                      // S7: residual quantisation, 1 / quantum
  float grid_z_lo;
  float Bc, err2_y, err2_z;
  float init_cov[5];
  float win_y, win_z, gate, max_sinphi, margin;
  float row_x[kMaxRows];
  float y_lo[kMaxRows], inv_by[kMaxRows], inv_bz[kMaxRows];
  float ny_hi[kMaxRows], nz_hi[kMaxRows];   // (float)(ny-1), (float)(nz-1): exact for < 2^24 bins
  int32_t ny[kMaxRows], nz[kMaxRows];
  int32_t bin_base[kMaxRows + 1];       // first bin of row r inside a sector
  int32_t cb_base[kMaxRows + 1];        // S1 level 1: first coarse bucket (row, z slab) of row r
  int32_t n_cb;                         // coarse buckets per sector
  int32_t slab_shift;                   // S1 level 1: log2 of the z slices per coarse bucket
  float hy_up[kMaxRows], hz_up[kMaxRows], hy_dn[kMaxRows], hz_dn[kMaxRows], nf_cut[kMaxRows];
  NfConst nf[kMaxRows];                 // S2 per-row constants (host-filled in tpcca_create)
};

// One sector's input arrays (device pointers; copies in the workspace or borrowed) and its place
// in the concatenated sorted arrays.
struct SectorDesc {
  const float* y;
  const float* z;
  const uint16_t* row;
  int32_t n;          // clusters in the sector
  int32_t off;        // first global position of the sector in the concatenated arrays
  int32_t tile256;    // first 256-cluster tile of the sector
  int32_t tile2048;   // first 2048-cluster tile of the sector
  int32_t pad[2];
};

// Device counters / status, mirrored to pinned host memory at the end of a run.
struct DevStatus {
  int32_t err_range;       // some cluster had row >= n_rows
  int32_t err_capacity;    // n_start exceeded max_start_hits
  int32_t err_select;      // S6: a sector holds 2^23 or more tracks (ownership key overflow)
  uint32_t n_big;          // S1 coarse buckets too large for the shared-memory sort
  int32_t n_start;         // total start hits
  int32_t work_counter[8]; // S5 dynamic work distribution: one counter per kernel mode (index 1..4)
  int32_t start_off[kMaxSectors + 1];   // first start-hit slot of each sector
  int32_t trk_off[kMaxSectors + 1];     // first track of each sector
  int64_t hit_off[kMaxSectors + 1];     // first hit of each sector (global CSR base)
  unsigned long long work[5];           // S5 work counters: propagations, updates, gates, searches, candidates
  int32_t sel_off[kMaxSectors + 1];     // S6: first selected track of each sector
  int64_t sel_hit_off[kMaxSectors + 1]; // S6: first hit of each sector in the selected hit CSR
};

// ---- S1 key: by = clamp(floor((y - y_lo) * inv_bin_y), 0, ny - 1) ------------
__device__ __forceinline__ int bin_coord(float v, float lo, float inv, float hi) {
  float t = __fmul_rn(__fsub_rn(v, lo), inv);
  float f = floorf(t);
  f = f < 0.0f ? 0.0f : f;
  f = f > hi ? hi : f;
  return (int)f;
}

// Same value as bin_coord for every input (floor + convert in one instruction, integer clamps);
// used where the bin is only a search range (S2, S5), never for the S1 key itself.
__device__ __forceinline__ int bin_range(float v, float lo, float inv, int hi) {
  const int b = __float2int_rd(__fmul_rn(__fsub_rn(v, lo), inv));
  return min(max(b, 0), hi);
}

// ---- block-wide exclusive scan over one int per thread (blockDim multiple of 32, <= 1024) ----
template <class T>
__device__ __forceinline__ T block_exclusive_scan(T v, T* warp_sums /*[32] shared*/, T& total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  T inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    T t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) warp_sums[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    T w = lane < nw ? warp_sums[lane] : (T)0;
    T winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      T t = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += t;
    }
    warp_sums[lane] = winc - w;           // exclusive prefix of the warp sums
    if (lane == 31) warp_sums[32] = winc; // total
  }
  __syncthreads();
  T res = warp_sums[wid] + inc - v;
  total = warp_sums[32];
  __syncthreads();
  return res;
}

}  // namespace tpcca
