// S5 tracklet construction + fp32 Kalman helix fit.
// One tracklet per thread; the three phases (A follow links, B extrapolate up, C refit down) are
// folded into ONE loop over row steps so that the lanes of a warp, which sit in different phases,
// still share the propagate / search / update instruction stream.
#pragma once
#include "k_links.cuh"

namespace tpcca {

// Kalman state: plane x, parameters p = (y, z_rel, sin phi, dz/ds, q/pT), covariance lower
// triangle c_ij (i >= j).  Every operation below is one IEEE binary32 operation in exactly the
// order DESIGN.md 3.5 writes it (the library is compiled with --fmad=false; the _rn intrinsics
// are used where a contraction would otherwise be tempting for the compiler).
struct KF {
  float x;
  float p0, p1, p2, p3, p4;
  float c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
  float chi2;
  int n;
};

struct KFConst {
  float Bc, err2_y, err2_z, max_sinphi, c24, c640, c12;
  float ic0, ic1, ic2, ic3, ic4;
};

__device__ __forceinline__ void kf_reset_cov(KF& s, const KFConst& k) {
  s.c00 = k.ic0; s.c10 = 0.f; s.c11 = k.ic1; s.c20 = 0.f; s.c21 = 0.f; s.c22 = k.ic2;
  s.c30 = 0.f; s.c31 = 0.f; s.c32 = 0.f; s.c33 = k.ic3;
  s.c40 = 0.f; s.c41 = 0.f; s.c42 = 0.f; s.c43 = 0.f; s.c44 = k.ic4;
  s.chi2 = 0.f; s.n = 0;
}

// DESIGN.md 3.5 "Propagate to x2", in two parts so that a kernel can issue the loads of the search
// between them (the search window depends only on the transported mean): kf_prop_mean transports x,
// p0, p1, p2 and returns the Jacobian terms; kf_prop_cov transports the covariance.  Every operation
// and its order are those of the definition.  false (state untouched) if |sin phi| would exceed the limit.
struct KFJac { float n02, n04, n12, n13, n14, n24; bool moved; };

__device__ __forceinline__ bool kf_prop_mean(KF& s, float x2, const KFConst& K, KFJac& J) {
  const float dx = x2 - s.x;
  J.moved = false;
  if (dx == 0.0f) return true;
  const float k = s.p4 * K.Bc;
  const float ey = s.p2;
  const float ey2 = ey + k * dx;
  if (!(fabsf(ey) <= K.max_sinphi) || !(fabsf(ey2) <= K.max_sinphi)) return false;
  const float ex = sqrtf(1.0f - ey * ey);
  const float ex2 = sqrtf(1.0f - ey2 * ey2);
  const float sx = ex + ex2;
  const float sY = ey + ey2;
  const float tg = sY / sx;
  const float dy = dx * tg;
  const float d2 = dx * dx + dy * dy;
  float d = sqrtf(d2);
  if (dx < 0.0f) d = -d;
  const float tt = (k * k) * d2;
  const float dS = d * (1.0f + tt * (K.c24 + tt * K.c640));
  const float cc = 1.0f + (ex * ex2 + ey * ey2);
  J.n02 = (dx * cc) / ((sx * ex) * ex2);
  const float j4 = ((dx * dx) * cc) / (ex2 * (sx * sx));
  J.n04 = K.Bc * j4;
  J.n12 = s.p3 * ((dx * tg) / (ex * ex2));
  J.n13 = dS;
  J.n14 = (s.p3 * K.Bc) * ((dy / d) * j4 + ((k * d) * d2) * K.c12);
  J.n24 = K.Bc * dx;
  J.moved = true;
  s.p0 = s.p0 + dy;
  s.p1 = s.p1 + s.p3 * dS;
  s.p2 = ey2;
  s.x = x2;
  return true;
}

__device__ __forceinline__ void kf_prop_cov(KF& s, const KFJac& J) {
  if (!J.moved) return;
  const float n02 = J.n02, n04 = J.n04, n12 = J.n12, n13 = J.n13, n14 = J.n14, n24 = J.n24;
  // A = J*C (rows 0..2 differ from C), C' = A*J^T (lower triangle); terms left to right.
  const float A00 = s.c00 + n02 * s.c20 + n04 * s.c40;
  const float A02 = s.c20 + n02 * s.c22 + n04 * s.c42;
  const float A04 = s.c40 + n02 * s.c42 + n04 * s.c44;
  const float A10 = s.c10 + n12 * s.c20 + n13 * s.c30 + n14 * s.c40;
  const float A11 = s.c11 + n12 * s.c21 + n13 * s.c31 + n14 * s.c41;
  const float A12 = s.c21 + n12 * s.c22 + n13 * s.c32 + n14 * s.c42;
  const float A13 = s.c31 + n12 * s.c32 + n13 * s.c33 + n14 * s.c43;
  const float A14 = s.c41 + n12 * s.c42 + n13 * s.c43 + n14 * s.c44;
  const float A20 = s.c20 + n24 * s.c40;
  const float A21 = s.c21 + n24 * s.c41;
  const float A22 = s.c22 + n24 * s.c42;
  const float A23 = s.c32 + n24 * s.c43;
  const float A24 = s.c42 + n24 * s.c44;
  const float A30 = s.c30, A31 = s.c31, A32 = s.c32, A33 = s.c33, A34 = s.c43;
  const float A40 = s.c40, A41 = s.c41, A42 = s.c42, A43 = s.c43, A44 = s.c44;
  s.c00 = A00 + A02 * n02 + A04 * n04;
  s.c10 = A10 + A12 * n02 + A14 * n04;
  s.c20 = A20 + A22 * n02 + A24 * n04;
  s.c30 = A30 + A32 * n02 + A34 * n04;
  s.c40 = A40 + A42 * n02 + A44 * n04;
  s.c11 = A11 + A12 * n12 + A13 * n13 + A14 * n14;
  s.c21 = A21 + A22 * n12 + A23 * n13 + A24 * n14;
  s.c31 = A31 + A32 * n12 + A33 * n13 + A34 * n14;
  s.c41 = A41 + A42 * n12 + A43 * n13 + A44 * n14;
  s.c22 = A22 + A24 * n24;
  s.c32 = A32 + A34 * n24;
  s.c42 = A42 + A44 * n24;
  s.c33 = A33;
  s.c43 = A43;
  s.c44 = A44;
}

__device__ __forceinline__ bool kf_propagate(KF& s, float x2, const KFConst& K) {
  KFJac J;
  if (!kf_prop_mean(s, x2, K, J)) return false;
  kf_prop_cov(s, J);
  return true;
}

// DESIGN.md 3.5 "Update": two scalar updates, y (component 0) then z (component 1).
__device__ __forceinline__ void kf_update(KF& s, float ym, float zm, const KFConst& K) {
  {
    const float r = ym - s.p0;
    const float w = 1.0f / (s.c00 + K.err2_y);
    const float q0 = s.c00, q1 = s.c10, q2 = s.c20, q3 = s.c30, q4 = s.c40;
    const float k0 = q0 * w, k1 = q1 * w, k2 = q2 * w, k3 = q3 * w, k4 = q4 * w;
    s.p0 = s.p0 + k0 * r; s.p1 = s.p1 + k1 * r; s.p2 = s.p2 + k2 * r;
    s.p3 = s.p3 + k3 * r; s.p4 = s.p4 + k4 * r;
    s.c00 = s.c00 - k0 * q0;
    s.c10 = s.c10 - k1 * q0; s.c11 = s.c11 - k1 * q1;
    s.c20 = s.c20 - k2 * q0; s.c21 = s.c21 - k2 * q1; s.c22 = s.c22 - k2 * q2;
    s.c30 = s.c30 - k3 * q0; s.c31 = s.c31 - k3 * q1; s.c32 = s.c32 - k3 * q2; s.c33 = s.c33 - k3 * q3;
    s.c40 = s.c40 - k4 * q0; s.c41 = s.c41 - k4 * q1; s.c42 = s.c42 - k4 * q2; s.c43 = s.c43 - k4 * q3;
    s.c44 = s.c44 - k4 * q4;
    s.chi2 = s.chi2 + (r * r) * w;
  }
  {
    const float r = zm - s.p1;
    const float w = 1.0f / (s.c11 + K.err2_z);
    const float q0 = s.c10, q1 = s.c11, q2 = s.c21, q3 = s.c31, q4 = s.c41;
    const float k0 = q0 * w, k1 = q1 * w, k2 = q2 * w, k3 = q3 * w, k4 = q4 * w;
    s.p0 = s.p0 + k0 * r; s.p1 = s.p1 + k1 * r; s.p2 = s.p2 + k2 * r;
    s.p3 = s.p3 + k3 * r; s.p4 = s.p4 + k4 * r;
    s.c00 = s.c00 - k0 * q0;
    s.c10 = s.c10 - k1 * q0; s.c11 = s.c11 - k1 * q1;
    s.c20 = s.c20 - k2 * q0; s.c21 = s.c21 - k2 * q1; s.c22 = s.c22 - k2 * q2;
    s.c30 = s.c30 - k3 * q0; s.c31 = s.c31 - k3 * q1; s.c32 = s.c32 - k3 * q2; s.c33 = s.c33 - k3 * q3;
    s.c40 = s.c40 - k4 * q0; s.c41 = s.c41 - k4 * q1; s.c42 = s.c42 - k4 * q2; s.c43 = s.c43 - k4 * q3;
    s.c44 = s.c44 - k4 * q4;
    s.chi2 = s.chi2 + (r * r) * w;
  }
  s.n++;
}

// slot-space scratch of S5: one record of kTrkV 16-byte vectors per slot (written by the lane that completes the
// tracklet with 128-bit stores, read by k_track_gather) + the n_hits plane (0 = rejected) the scans read
constexpr int kTrkV = 7;    // (n_fit, first_row, last_row, -) (x_ref, z_ref, p0, p1) (p2, p3, p4, c00) ... (c43, c44, chi2, -)

constexpr int kS5Threads = 128;   // threads per block of k_tracklets
#ifndef TPCCA_S5_BPS
#define TPCCA_S5_BPS 5
#endif
#ifndef TPCCA_S5_BPS_A
#define TPCCA_S5_BPS_A 5
#endif
constexpr int kS5BlocksPerSMA = TPCCA_S5_BPS_A;   // ... of the phase-A kernel (no search code: fewer registers)
constexpr int kS5BlocksPerSM = TPCCA_S5_BPS;  // resident blocks per SM the kernel is compiled for (persistent grid)
#ifndef TPCCA_S5_REFILL
#define TPCCA_S5_REFILL 6
#endif
constexpr int kS5Refill = TPCCA_S5_REFILL;      // idle lanes of a warp that trigger a refill from the work counter
#ifndef TPCCA_S5_UNROLL
#define TPCCA_S5_UNROLL 5
#endif
constexpr int kS5Unroll = TPCCA_S5_UNROLL;   // candidate loads in flight per lane in the S5 search
#ifndef TPCCA_S5_SEARCH_BATCH
#define TPCCA_S5_SEARCH_BATCH 4
#endif
constexpr int kS5SearchBatch = TPCCA_S5_SEARCH_BATCH;   // phase-C1 lanes that wait for each other before a search is issued
constexpr int kSnapF = 22;        // floats of a saved Kalman state: x, p[5], c[15], chi2

// scalars of S5, passed by value (constant bank: no registers)
struct S5Params {
  float Bc, err2_y, err2_z, max_sinphi;
  float ic0, ic1, ic2, ic3, ic4;
  float win_y, win_z, gate, margin, grid_z_lo;
  int32_t n_rows, n_sectors, max_gap, min_hits, bins_per_sector;
};

// approximate reciprocal (one MUFU.RCP); used only to rank candidates and to pre-decide gates
// that are nowhere near the threshold -- every decision that could flip is taken on the exact form
__device__ __forceinline__ float rcp_fast(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// Gate of DESIGN.md 3.5: dist2 = ry^2 / wy + rz^2 / wz > gate, decided exactly.  The division-free
// estimate is within ~1e-6 relative of dist2, so it decides whenever it is more than 1e-4 relative
// away from the gate; otherwise (and for NaN / inf estimates) the defined expression is evaluated.
__device__ __forceinline__ bool gate_exceeded(float ry, float rz, float wy, float wz, float iwy, float iwz, float gate) {
  const float ry2 = ry * ry, rz2 = rz * rz;
  const float est = ry2 * iwy + rz2 * iwz;
  if (est > gate * 1.0001f + 1e-30f) return true;
  if (est < gate * 0.9999f - 1e-30f) return false;
  return (ry2 / wy + rz2 / wz) > gate;
}

// Exact search of S5: minimum d2 = ry^2 / wy + rz^2 / wz over the window, ties ->
// smallest original id.  Out of line: the kernel's ranking loop calls it only when two candidates
// are too close for its division-free ranking to separate.
__device__ __noinline__ int search_exact(float p0, float p1, float z_ref, float wy, float wz, float win_y, float win_z,
                                         const uint32_t* __restrict__ bp, int ny, int by0, int by1, int nsl,
                                         const float2* __restrict__ yz, const int32_t* __restrict__ ord,
                                         float& best_d2, float2& best_h, unsigned& n_cand) {
  int best = -1;
  best_d2 = 0.f;
  for (int k = 0; k < nsl; ++k) {
    const uint32_t e = __ldg(&bp[k * ny + by1 + 1]);
    for (uint32_t c = __ldg(&bp[k * ny + by0]); c < e; ++c) {
      const float2 h = __ldg(&yz[c]);
      const float ry = h.x - p0;
      const float rz = (h.y - z_ref) - p1;
      if (!(fabsf(ry) <= win_y && fabsf(rz) <= win_z)) continue;
      const float d2 = (ry * ry) / wy + (rz * rz) / wz;
      ++n_cand;
      if (best < 0 || d2 < best_d2 || (d2 == best_d2 && __ldg(&ord[c]) < __ldg(&ord[best]))) {
        best = (int)c; best_d2 = d2; best_h = h;
      }
    }
  }
  return best;
}

// ---- K5a ---------------------------------------------------------------------------------------
// One tracklet per thread.  The three phases (A follow links, B extrapolate up, C refit down) are
// folded into ONE loop over row steps, so lanes in different phases share the propagate / search /
// update instruction stream.  A lane that finishes its tracklet goes idle; as soon as kS5Refill
// lanes of the warp are idle (or no lane is active) the warp takes that many new start hits from
// the global work counter, so warps never wait for their longest tracklet.
// The phase-C snapshot ("state right after the last update") lives in registers while it equals
// the running state and is parked in shared memory the moment the running state moves on without
// an update, which keeps the register count at one Kalman state per lane.
// The kernel is compiled in four modes and launched four times: MODE_A runs phase A
// for every start hit, MODE_B phase B, MODE_C1 phase C down to the start row (hits known: updates, a search
// only on gap rows), MODE_C2 phase C below the start row (a search every row).  A lane whose tracklet leaves the kernel's phase
// parks the tracklet (Kalman state + bookkeeping, kHsF floats and kHsI ints, indexed by the work
// index so that the lanes refilled together store and load neighbouring words) and takes new work.
// Per lane the sequence of operations is exactly that of the single loop; what changes is which
// lanes share a warp: link followers (no search), extrapolators (a search every row) and refitters
// no longer wait for each other's code.
enum { MODE_A = 1, MODE_B = 2, MODE_C1 = 3, MODE_C2 = 4 };
// parked tracklet: one record of kHsV 16-byte vectors, indexed by the work index; a tracklet bound for phase C
// only fills the first four: (x, p0, p1, p2) (p3, p4, z_ref, phase) (top, top_hit, n_hits, first) (r0, n, r, cur)
// (gap, c00, c10, c11) (c20, c21, c22, c30) (c31, c32, c33, c40) (c41, c42, c43, c44) (chi2, -, -, -)
constexpr int kHsV = 9;

template <int MODE>
__global__ void __launch_bounds__(kS5Threads, MODE == MODE_A ? kS5BlocksPerSMA : kS5BlocksPerSM)
k_tracklets(const DevTables* __restrict__ T, const SectorDesc* __restrict__ sec,
            DevStatus* __restrict__ st, const S5Params P, const float2* __restrict__ syz,
            const uint32_t* __restrict__ bin_start, const int32_t* __restrict__ order,
            const int32_t* __restrict__ link_up, const int4* __restrict__ perm, int32_t cap,
            int32_t* __restrict__ hits /*[cap][n_rows]*/, float4* __restrict__ trk_v /*[cap][kTrkV]*/,
            int32_t* __restrict__ trk_n /*[cap]*/, float4* __restrict__ hs /*[cap][kHsV]*/) {
  __shared__ float t_x[kMaxRows], t_ylo[kMaxRows], t_iby[kMaxRows], t_ibz[kMaxRows];
  __shared__ int32_t t_nyh[kMaxRows], t_nzh[kMaxRows], t_ny[kMaxRows], t_base[kMaxRows];
  __shared__ int s_sec_off[kMaxSectors + 1];
  __shared__ float s_snap[kSnapF][kS5Threads];
  const int n_rows = P.n_rows, ns = P.n_sectors;
  for (int r = threadIdx.x; r < n_rows; r += blockDim.x) {
    t_x[r] = T->row_x[r]; t_ylo[r] = T->y_lo[r]; t_iby[r] = T->inv_by[r]; t_nyh[r] = T->ny[r] - 1;
    t_ibz[r] = T->inv_bz[r]; t_nzh[r] = T->nz[r] - 1; t_ny[r] = T->ny[r]; t_base[r] = T->bin_base[r];
  }
  for (int i = threadIdx.x; i <= ns; i += blockDim.x) s_sec_off[i] = sec[i].off;
  __syncthreads();
  if (st->err_capacity || st->err_range) return;
  const int n_start = st->n_start;
  KFConst K;
  K.Bc = P.Bc; K.err2_y = P.err2_y; K.err2_z = P.err2_z; K.max_sinphi = P.max_sinphi;
  K.c24 = (float)(1.0 / 24.0); K.c640 = (float)(3.0 / 640.0); K.c12 = (float)(1.0 / 12.0);
  K.ic0 = P.ic0; K.ic1 = P.ic1; K.ic2 = P.ic2; K.ic3 = P.ic3; K.ic4 = P.ic4;
  const float my = P.win_y + P.margin, mz = P.win_z + P.margin;
  const uint32_t nbp1 = (uint32_t)P.bins_per_sector + 1u;
  const int lane = threadIdx.x & 31;
  const int tid = threadIdx.x;
  unsigned w_prop = 0, w_upd = 0, w_gate = 0, w_search = 0, w_cand = 0;   // work counters

  enum { PH_A = 0, PH_B = 1, PH_C = 2, PH_IDLE = 3, PH_C2 = 4 };   // PH_C2: parked marker only (phase C below the start row)
  // ---- per-lane tracklet state ---------------------------------------------------------------
  int phase = PH_IDLE;
  bool drained = false;      // warp-uniform: the work counter ran out
  int wi = 0;                // work index of the lane's tracklet (parking slot)
  int slot = 0, r = 0, cur = -1, top = 0, top_hit = -1, gap = 0, n_hits = 0, first = 0, r0 = 0;
  int nxt_pre = -1;          // MODE_A / MODE_C1: hit of the next row (read one step ahead) ...
  float2 h_pre = make_float2(0.f, 0.f);   // ... and the cluster of row r (loaded one step ahead)
  bool fresh = false;        // running state == snapshot (last operation was a phase-C update)
  bool saved = false;        // snapshot parked in shared memory
  float z_ref = 0.f;
  int off = 0;               // first sorted position of the lane's sector in the concatenated arrays
  uint32_t bs_off = 0;       // first bin_start entry of the lane's sector (fits 32 bits: tpcca_create checks)
  KF f;
  f.x = 0.f; f.p0 = f.p1 = f.p2 = f.p3 = f.p4 = 0.f;
  kf_reset_cov(f, K);

  auto save_snap = [&]() {
    s_snap[0][tid] = f.x; s_snap[1][tid] = f.p0; s_snap[2][tid] = f.p1; s_snap[3][tid] = f.p2;
    s_snap[4][tid] = f.p3; s_snap[5][tid] = f.p4;
    s_snap[6][tid] = f.c00; s_snap[7][tid] = f.c10; s_snap[8][tid] = f.c11; s_snap[9][tid] = f.c20;
    s_snap[10][tid] = f.c21; s_snap[11][tid] = f.c22; s_snap[12][tid] = f.c30; s_snap[13][tid] = f.c31;
    s_snap[14][tid] = f.c32; s_snap[15][tid] = f.c33; s_snap[16][tid] = f.c40; s_snap[17][tid] = f.c41;
    s_snap[18][tid] = f.c42; s_snap[19][tid] = f.c43; s_snap[20][tid] = f.c44; s_snap[21][tid] = f.chi2;
  };
  int snap_n = 0;            // f.n at the time of the snapshot
  // emit the tracklet of this lane into slot space and go idle
  auto finish = [&]() {
    if (fresh) { save_snap(); snap_n = f.n; saved = true; }
    const bool accept = (n_hits >= P.min_hits) && saved;
    trk_n[slot] = accept ? n_hits : 0;
    if (accept) {
      float4* o = trk_v + (size_t)slot * kTrkV;
      const float* sn = &s_snap[0][tid];
      auto S = [&](int k) { return sn[k * kS5Threads]; };
      o[0] = make_float4(__int_as_float(snap_n), __int_as_float(first), __int_as_float(top), 0.f);
      o[1] = make_float4(S(0), z_ref, S(1), S(2));
      o[2] = make_float4(S(3), S(4), S(5), S(6));
      o[3] = make_float4(S(7), S(8), S(9), S(10));
      o[4] = make_float4(S(11), S(12), S(13), S(14));
      o[5] = make_float4(S(15), S(16), S(17), S(18));
      o[6] = make_float4(S(19), S(20), S(21), 0.f);
    }
    phase = PH_IDLE;
  };

  // park the tracklet for the next kernel and go idle.  A tracklet bound for phase C carries only x, p
  // and z_ref: the covariance reset, r = top, cur = top_hit and gap = 0 of the phase change are applied by
  // the phase-C1 kernel when it loads the tracklet.
  auto park = [&]() {
    float4* o = hs + (size_t)wi * kHsV;
    auto I = [](int v) { return __int_as_float(v); };
    o[0] = make_float4(f.x, f.p0, f.p1, f.p2);
    o[1] = make_float4(f.p3, f.p4, z_ref, I(phase));
    o[2] = make_float4(I(top), I(top_hit), I(n_hits), I(first));
    o[3] = make_float4(I(r0), I(f.n), I(r), I(cur));
    if (phase != PH_C) {
      o[4] = make_float4(I(gap), f.c00, f.c10, f.c11);
      o[5] = make_float4(f.c20, f.c21, f.c22, f.c30);
      o[6] = make_float4(f.c31, f.c32, f.c33, f.c40);
      o[7] = make_float4(f.c41, f.c42, f.c43, f.c44);
      o[8] = make_float4(f.chi2, 0.f, 0.f, 0.f);
    }
    phase = PH_IDLE;
  };

  for (;;) {
    // ---- refill idle lanes from the work counter ---------------------------------------------
    const unsigned idle = __ballot_sync(0xffffffffu, phase == PH_IDLE);
    if (idle == 0xffffffffu && drained) break;
    if (!drained && (__popc(idle) >= kS5Refill || idle == 0xffffffffu)) {
      const int n_idle = __popc(idle);
      int base = 0;
      if (lane == 0) base = atomicAdd(&st->work_counter[MODE], n_idle);
      base = __shfl_sync(0xffffffffu, base, 0);
      if (base + n_idle >= n_start) drained = true;
      if (phase == PH_IDLE) {
        const int my_w = base + __popc(idle & ((1u << lane) - 1u));
        if (my_w < n_start) {
          wi = my_w;
          const int4 pr = __ldg(&perm[my_w]);   // slot, start row | sector << 16, start hit
          slot = pr.x;
          const int s = pr.y >> 16;
          off = s_sec_off[s];
          bs_off = (uint32_t)s * nbp1;
          if (MODE == MODE_A) {
            const int c0 = pr.z;
            r0 = pr.y & 0xffff;
            const int c1 = __ldg(&link_up[off + c0]);
            const float2 h0 = __ldg(&syz[off + c0]), h1 = __ldg(&syz[off + c1]);
            z_ref = h0.y;
            const float dx = t_x[r0 + 1] - t_x[r0];
            const float dy = h1.x - h0.x;
            const float dz = h1.y - z_ref;
            const float d = sqrtf(dx * dx + dy * dy);
            f.x = t_x[r0];
            f.p0 = h0.x; f.p1 = 0.f; f.p2 = dy / d; f.p3 = dz / d; f.p4 = 0.f;
            kf_reset_cov(f, K);
            phase = PH_A; r = r0; cur = c0; top = r0; top_hit = c0; gap = 0; n_hits = 0; first = r0;
            h_pre = h0; nxt_pre = c1;
            fresh = false; saved = false;
          } else {
            const float4* o = hs + (size_t)wi * kHsV;
            auto I = [](float v) { return __float_as_int(v); };
            const float4 v0 = o[0], v1 = o[1], v2 = o[2], v3 = o[3];
            float4 v4, v5, v6, v7, v8;
            if (MODE != MODE_C1) { v4 = o[4]; v5 = o[5]; v6 = o[6]; v7 = o[7]; v8 = o[8]; }   // issued before the phase test
            const int ph = I(v1.w);
            if (ph == (MODE == MODE_B ? PH_B : (MODE == MODE_C1 ? PH_C : PH_C2))) {   // others are not this kernel's
              f.x = v0.x; f.p0 = v0.y; f.p1 = v0.z; f.p2 = v0.w; f.p3 = v1.x; f.p4 = v1.y; z_ref = v1.z;
              top = I(v2.x); top_hit = I(v2.y); n_hits = I(v2.z); first = I(v2.w); r0 = I(v3.x);
              if (MODE == MODE_C1) {          // the phase change A/B -> C is completed here
                kf_reset_cov(f, K); gap = 0; r = top; cur = top_hit;
                {
                  const int32_t* line = hits + (size_t)slot * n_rows;
                  nxt_pre = (r - 1 >= r0) ? line[r - 1] : -1;
                  h_pre = cur >= 0 ? __ldg(&syz[off + cur]) : make_float2(0.f, 0.f);
                }
              } else {
                f.n = I(v3.y); r = I(v3.z); cur = I(v3.w); gap = I(v4.x);
                f.c00 = v4.y; f.c10 = v4.z; f.c11 = v4.w; f.c20 = v5.x; f.c21 = v5.y; f.c22 = v5.z; f.c30 = v5.w;
                f.c31 = v6.x; f.c32 = v6.y; f.c33 = v6.z; f.c40 = v6.w; f.c41 = v7.x; f.c42 = v7.y; f.c43 = v7.z; f.c44 = v7.w;
                f.chi2 = v8.x;
              }
              phase = (MODE == MODE_C2) ? (int)PH_C : ph;
              // C1 always hands over right after the update on the start row: running state == snapshot
              fresh = (MODE == MODE_C2); saved = false;
            }
          }
        }
      }
    }
    // ---- one row step.  Every lane walks the same sequence of blocks (no early exits), with
    // warp syncs in front of the heavy ones, so the warp executes propagate / search / update
    // together whatever phases its lanes are in.  Phase changes are recorded in `ev` and applied
    // once at the end of the step. ----------------------------------------------------------------
    enum { EV_NONE = 0, EV_TO_C = 1, EV_FINISH = 2 };
    const bool alive = phase != PH_IDLE;
    int ev = EV_NONE;
    int32_t* hcol = hits + (size_t)slot * n_rows;   // the tracklet's hit per row: one contiguous line per tracklet
    int cand = -1;                        // >= 0: cluster to use on this row; -1: none known
    int nxt = -1;                         // candidate of the next row (loaded early)
    int nn = -1;                          // MODE_C1: candidate of the row after the next
    float2 hn = make_float2(0.f, 0.f);    // MODE_C1: cluster of the next row
    float2 h = make_float2(0.f, 0.f);
    float xr = f.x;
    if (alive) {
      cand = cur;
      if (MODE == MODE_C1) {
        // refit over known hits: the hit of the next row and the cluster of this row were read one step
        // ahead, the loads issued here are consumed at the end of the step (their latency is off the path)
        h = h_pre; nxt = nxt_pre;
        if (r - 2 >= r0) nn = hcol[r - 2];
        if (nxt >= 0) hn = __ldg(&syz[off + nxt]);
      } else if (MODE == MODE_A) {
        // link following: the chain is walked one link ahead of the fit (same reason)
        h = h_pre; nxt = nxt_pre;
        if (nxt >= 0) { nn = __ldg(&link_up[off + nxt]); hn = __ldg(&syz[off + nxt]); }
      } else {
        if (cand >= 0) h = __ldg(&syz[off + cand]);
        if (phase == PH_C && r - 1 >= r0) nxt = hcol[r - 1];
      }
      xr = t_x[r];
      if (phase == PH_C && fresh && cand < 0) { save_snap(); snap_n = f.n; saved = true; fresh = false; }
      w_prop += (xr != f.x) ? 1u : 0u;
    }
    __syncwarp();
    bool go = false;                      // the lane carries on with this row
    // kernels that search every row: the bin_start loads of the search are issued between the two
    // halves of the propagation (the window depends only on the transported mean), so their latency
    // overlaps the covariance transport
    constexpr bool kEarly = (MODE == MODE_B || MODE == MODE_C2);
    uint32_t c0 = 0, e0 = 0, c1 = 0, e1 = 0, c2 = 0, e2 = 0;
    int nsl = 0;
    if (alive) {
      KFJac J;
      go = kf_prop_mean(f, xr, K, J);
      if (!go) ev = (phase == PH_C) ? EV_FINISH : EV_TO_C;
      if (kEarly && go && cand < 0 && (phase == PH_B || f.n >= 2)) {
        const float ylo = t_ylo[r], iby = t_iby[r], ibz = t_ibz[r];
        const int nyh = t_nyh[r], nzh = t_nzh[r], ny = t_ny[r];
        const float zc = z_ref + f.p1;
        const int by0 = bin_range(f.p0 - my, ylo, iby, nyh), by1 = bin_range(f.p0 + my, ylo, iby, nyh);
        const int bz0 = bin_range(zc - mz, P.grid_z_lo, ibz, nzh), bz1 = bin_range(zc + mz, P.grid_z_lo, ibz, nzh);
        const uint32_t* bp = bin_start + (bs_off + (uint32_t)(t_base[r] + bz0 * ny));
        nsl = bz1 - bz0 + 1;
        c0 = __ldg(&bp[by0]); e0 = __ldg(&bp[by1 + 1]);
        if (nsl > 1) { c1 = __ldg(&bp[ny + by0]); e1 = __ldg(&bp[ny + by1 + 1]); }
        if (nsl > 2) { c2 = __ldg(&bp[2 * ny + by0]); e2 = __ldg(&bp[2 * ny + by1 + 1]); }
      }
      if (go) kf_prop_cov(f, J);
    }
    bool took = false, is_new = false, need_search = false;
    const float wy = f.c00 + K.err2_y;
    const float wz = f.c11 + K.err2_z;
    const float iwy = rcp_fast(wy), iwz = rcp_fast(wz);   // ranking only, never a decision on its own
    if (go) {
      if (phase == PH_A) {
        bool ok = true;
        if (f.n >= 2) {
          ++w_gate;
          ok = !gate_exceeded(h.x - f.p0, (h.y - z_ref) - f.p1, wy, wz, iwy, iwz, P.gate);
        }
        if (ok) { took = true; is_new = true; }
        else { phase = PH_B; gap = 0; cur = -1; go = false; }   // state already sits on row r (dx = 0 next)
      } else if (cand >= 0) {
        took = true;                      // phase C, row already holds a hit: no gate
      } else {
        need_search = (phase == PH_B) || (f.n >= 2);
      }
    }
    __syncwarp();
    if (MODE == MODE_C1) {
      // Refit over known hits: only the few lanes on a hit-less row search, and each such step would issue the whole
      // search code for one or two lanes (23 % of this kernel's instructions ran at < 4 active lanes).  A lane that
      // needs a search therefore WAITS on its row (the state already sits there: repeating the step is a no-op up to
      // this point) until kS5SearchBatch lanes of the warp wait, or every live lane does.
      const unsigned want = __ballot_sync(0xffffffffu, need_search);
      if (want) {
        const unsigned live = __ballot_sync(0xffffffffu, alive);
        if (__popc(want) < kS5SearchBatch && want != live) {
          if (need_search) { need_search = false; go = false; }
        }
      }
    }
    if (MODE != MODE_A && need_search) {
      // search: best cluster of row r in the tc window around the prediction
      const float yc = f.p0;
      const float zc = z_ref + f.p1;
      const float ylo = t_ylo[r], iby = t_iby[r], ibz = t_ibz[r];
      const int nyh = t_nyh[r], nzh = t_nzh[r];
      const int by0 = bin_range(yc - my, ylo, iby, nyh), by1 = bin_range(yc + my, ylo, iby, nyh);
      const int bz0 = bin_range(zc - mz, P.grid_z_lo, ibz, nzh), bz1 = bin_range(zc + mz, P.grid_z_lo, ibz, nzh);
      const int ny = t_ny[r];
      const uint32_t* bp = bin_start + (bs_off + (uint32_t)(t_base[r] + bz0 * ny));
      const float2* yz = syz + off;
      ++w_search;
      // The candidates of the (at most three) z slices are walked as ONE loop over a flat index,
      // so the trip count of the warp is the largest candidate count of a lane, not the sum of the
      // largest runs.  Ranking is done on d2~ = ry^2 * (1/wy)~ + rz^2 * (1/wz)~ (no division): d2~
      // is within a few ulp of the defined d2, so the smallest d2~ is the smallest d2 unless the
      // runner-up is within 2e-5 relative; then (ties, duplicates), and for windows of more than
      // three slices, the exact loop decides.
      if (!kEarly) {
        nsl = bz1 - bz0 + 1;
        c0 = __ldg(&bp[by0]); e0 = __ldg(&bp[by1 + 1]);
        if (nsl > 1) { c1 = __ldg(&bp[ny + by0]); e1 = __ldg(&bp[ny + by1 + 1]); }
        if (nsl > 2) { c2 = __ldg(&bp[2 * ny + by0]); e2 = __ldg(&bp[2 * ny + by1 + 1]); }
      }
      const int n0 = (int)(e0 - c0), n01 = n0 + (int)(e1 - c1), total = nsl > 3 ? 0 : n01 + (int)(e2 - c2);
      const uint32_t o1 = c1 - (uint32_t)n0, o2 = c2 - (uint32_t)n01;   // flat index i -> cluster o + i
      float a1 = __int_as_float(0x7f800000), a2 = a1;
      int best = -1;
      // kS5Unroll candidate loads are issued together: the loop is bound by load latency
      for (int i = 0; i < total; i += kS5Unroll) {
        uint32_t cc[kS5Unroll];
        float2 hh[kS5Unroll];
#pragma unroll
        for (int k = 0; k < kS5Unroll; ++k) {
          const int j = min(i + k, total - 1);
          cc[k] = (uint32_t)j + (j < n0 ? c0 : (j < n01 ? o1 : o2));
        }
#pragma unroll
        for (int k = 0; k < kS5Unroll; ++k) hh[k] = __ldg(&yz[cc[k]]);
#pragma unroll
        for (int k = 0; k < kS5Unroll; ++k) {
          const float ry = hh[k].x - f.p0;
          const float rz = (hh[k].y - z_ref) - f.p1;
          if (i + k < total && fabsf(ry) <= P.win_y && fabsf(rz) <= P.win_z) {
            const float da = (ry * ry) * iwy + (rz * rz) * iwz;
            ++w_cand;
            if (da < a1) { a2 = a1; a1 = da; best = (int)cc[k]; }
            else a2 = fminf(a2, da);
          }
        }
      }
      if (best >= 0 || nsl > 3) {
        bool pass;
        if (nsl > 3 || !(a2 > a1 * 1.00002f + 1e-30f)) {
          float best_d2;
          unsigned n_cand = 0;
          best = search_exact(f.p0, f.p1, z_ref, wy, wz, P.win_y, P.win_z, bp, ny, by0, by1, nsl, yz, order + off, best_d2, h, n_cand);
          if (nsl > 3) w_cand += n_cand;
          pass = best >= 0 && best_d2 <= P.gate;
        } else {
          h = __ldg(&yz[best]);
          pass = !gate_exceeded(h.x - f.p0, (h.y - z_ref) - f.p1, wy, wz, iwy, iwz, P.gate);
        }
        if (pass) { cand = best; took = true; is_new = true; }
      }
    }
    __syncwarp();
    if (go) {
      if (took) {
        kf_update(f, h.x, h.y - z_ref, K);
        ++w_upd;
        if (is_new) { hcol[r] = cand; ++n_hits; }
        if (phase == PH_C) {
          fresh = true; saved = false;
          if (is_new) { gap = 0; if (r < first) first = r; }
        } else {
          top = r; top_hit = cand; gap = 0;
        }
      } else if (phase == PH_B) {
        hcol[r] = -1;
        if (++gap > P.max_gap) { ev = EV_TO_C; go = false; }
      } else if (r < r0) {                // phase C below the start hit
        hcol[r] = -1;
        if (++gap > P.max_gap) { ev = EV_FINISH; go = false; }
      }
    }
    // ---- advance to the next row -------------------------------------------------------------
    if (go) {
      if (phase == PH_A) { cur = nxt; ++r; if (MODE == MODE_A) { nxt_pre = nn; h_pre = hn; } if (cur == -1) { phase = PH_B; gap = 0; } }
      else if (phase == PH_B) ++r;
      else { cur = nxt; --r; if (MODE == MODE_C1) { nxt_pre = nn; h_pre = hn; } }
      if (phase == PH_B && r >= n_rows) ev = EV_TO_C;
      if (phase == PH_C && r < 0) ev = EV_FINISH;
    }
    // A tracklet that leaves the kernel's phase is parked (the record is a few 128-bit stores), a complete one
    // is emitted; either way the lane goes idle.
    if (ev == EV_TO_C) {                  // phases A / B only, i.e. MODE_A / MODE_B: the tracklet leaves the kernel
      phase = PH_C; park();               // (covariance reset, r, cur, gap: applied by MODE_C1 on load)
    } else if (ev == EV_FINISH) {
      finish();
    }
    if (MODE == MODE_A && phase == PH_B) park();
    if (MODE == MODE_C1 && phase == PH_C && r < r0) { phase = PH_C2; park(); }
  }
  // work counters: one atomic per warp and counter
  unsigned long long w[5] = {w_prop, w_upd, w_gate, w_search, w_cand};
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    unsigned long long v = w[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0 && v) atomicAdd(&st->work[i], v);
  }
}

// ---- K5b: per-tile (1024 slots) sums of (accepted, n_hits) ------------------------------------
__global__ void __launch_bounds__(1024)
k_track_tile_sums(const DevStatus* __restrict__ st, const int32_t* __restrict__ trk_n, int2* __restrict__ tile_cnt) {
  __shared__ int ws[33];
  const int n_start = st->err_capacity ? 0 : st->n_start;
  const int slot = blockIdx.x * 1024 + threadIdx.x;
  const int nh = slot < n_start ? trk_n[slot] : 0;
  int ta, tb;
  block_exclusive_scan<int>(nh > 0 ? 1 : 0, ws, ta);
  block_exclusive_scan<int>(nh, ws, tb);
  if (threadIdx.x == 0) tile_cnt[blockIdx.x] = make_int2(ta, tb);
}

// ---- K5c': sector bases of the track table and of the hit CSR ---------------------------------
__global__ void k_track_sector_bases(const DevTables* __restrict__ T, DevStatus* __restrict__ st,
                                     const int32_t* __restrict__ trk_n, const longlong2* __restrict__ tile_off,
                                     const int64_t* __restrict__ tot) {
  const int ns = T->n_sectors;
  const int s = threadIdx.x;
  if (s > ns) return;
  const int n_start = st->err_capacity ? 0 : st->n_start;
  const int slot = st->err_capacity ? 0 : st->start_off[s];
  if (slot >= n_start) { st->trk_off[s] = (int32_t)tot[0]; st->hit_off[s] = tot[1]; return; }
  const int t = slot >> 10;
  long long a = tile_off[t].x, b = tile_off[t].y;
  for (int q = t << 10; q < slot; ++q) { const int nh = trk_n[q]; a += nh > 0; b += nh; }
  st->trk_off[s] = (int32_t)a;
  st->hit_off[s] = b;
}

// ---- K5d: gather accepted tracklets into the track table + hit CSR (start-hit order) ----------
struct TrackOut {
  float *x_ref, *z_ref, *par, *cov, *chi2;
  int32_t *n_hits, *n_fit, *first_row, *last_row, *start_hit, *hit_offset, *hit_idx;
};

__global__ void __launch_bounds__(1024)
k_track_gather(const DevTables* __restrict__ T, const DevStatus* __restrict__ st,
               const int32_t* __restrict__ start_hit, int32_t cap, const int32_t* __restrict__ hits,
               const float4* __restrict__ trk_v, const int32_t* __restrict__ trk_n,
               const longlong2* __restrict__ tile_off, TrackOut o, int32_t* __restrict__ slot_trk /*[cap]: slot -> track, -1*/) {
  __shared__ int ws[33];
  const int ns = T->n_sectors, n_rows_g = T->n_rows;
  const int n_start = st->err_capacity ? 0 : st->n_start;
  const int slot = blockIdx.x * 1024 + threadIdx.x;
  const int nh = slot < n_start ? trk_n[slot] : 0;
  int ta, tb;
  const int ea = block_exclusive_scan<int>(nh > 0 ? 1 : 0, ws, ta);
  const int eb = block_exclusive_scan<int>(nh, ws, tb);
  const bool valid = slot < n_start;
  // sector of the slot
  int s = 0;
  if (valid) {
    int lo = 0, hi = ns - 1;
    while (lo < hi) { int mid = (lo + hi + 1) >> 1; if (st->start_off[mid] <= slot) lo = mid; else hi = mid - 1; }
    s = lo;
  }
  const long long t = tile_off[blockIdx.x].x + ea;       // global track index
  const long long h = tile_off[blockIdx.x].y + eb;       // global hit index
  int first = 0, last = -1;
  if (valid) {
    slot_trk[slot] = nh > 0 ? (int32_t)t : -1;
    const long long hloc = h - st->hit_off[s];
    // hit_offset of sector s lives at [trk_off[s] + s, trk_off[s+1] + s + 1)
    if (nh > 0) {
      const size_t cs = (size_t)cap;
      o.hit_offset[t + s] = (int32_t)hloc;
      const float4* v = trk_v + (size_t)slot * kTrkV;
      const float4 v0 = v[0], v1 = v[1], v2 = v[2], v3 = v[3], v4 = v[4], v5 = v[5], v6 = v[6];
      o.x_ref[t] = v1.x;
      o.z_ref[t] = v1.y;
      const float par[5] = {v1.z, v1.w, v2.x, v2.y, v2.z};
      const float cov[15] = {v2.w, v3.x, v3.y, v3.z, v3.w, v4.x, v4.y, v4.z, v4.w, v5.x, v5.y, v5.z, v5.w, v6.x, v6.y};
#pragma unroll
      for (int i = 0; i < 5; ++i) o.par[i * cs + t] = par[i];
#pragma unroll
      for (int i = 0; i < 15; ++i) o.cov[i * cs + t] = cov[i];
      o.chi2[t] = v6.z;
      o.n_hits[t] = nh;
      o.n_fit[t] = __float_as_int(v0.x);
      first = __float_as_int(v0.y); last = __float_as_int(v0.z);
      o.first_row[t] = first;
      o.last_row[t] = last;
      o.start_hit[t] = start_hit[slot];
    }
    // closing entry of each sector's hit_offset: written by the last slot of the sector (empty
    // sectors are closed by k_track_close_empty)
    if (slot + 1 == st->start_off[s + 1] || slot + 1 == n_start) {
      const long long tend = t + (nh > 0 ? 1 : 0);
      o.hit_offset[tend + s] = (int32_t)(hloc + nh);
    }
  }
  // hit CSR: the warp copies the hit line of each of its accepted tracklets together (coalesced
  // 128-byte reads of the tracklet's line, ballot compaction of the rows that hold a hit)
  const int lane = threadIdx.x & 31;
  unsigned todo = __ballot_sync(0xffffffffu, valid && nh > 0);
  while (todo) {
    const int src = __ffs(todo) - 1;
    todo &= todo - 1;
    const int sl = __shfl_sync(0xffffffffu, slot, src);
    const int f0 = __shfl_sync(0xffffffffu, first, src), l0 = __shfl_sync(0xffffffffu, last, src);
    long long w = __shfl_sync(0xffffffffu, h, src);
    const int32_t* line = hits + (size_t)sl * n_rows_g;
    // the loads of up to kG x 32 rows are issued together (one memory latency per tracklet, not one per 32 rows)
    constexpr int kG = 5;
    for (int r0 = f0; r0 <= l0; r0 += 32 * kG) {
      int cc[kG];
#pragma unroll
      for (int q = 0; q < kG; ++q) {
        const int r = r0 + 32 * q + lane;
        cc[q] = r <= l0 ? __ldcs(&line[r]) : -1;
      }
#pragma unroll
      for (int q = 0; q < kG; ++q) {
        if (r0 + 32 * q > l0) break;             // warp-uniform
        const unsigned m = __ballot_sync(0xffffffffu, cc[q] != -1);
        if (cc[q] != -1) o.hit_idx[w + __popc(m & ((1u << lane) - 1u))] = cc[q];
        w += __popc(m);
      }
    }
  }
}

// sectors without start hits still own a one-entry hit_offset = {0}
__global__ void k_track_close_empty(const DevTables* __restrict__ T, const DevStatus* __restrict__ st, TrackOut o) {
  const int ns = T->n_sectors;
  const int s = threadIdx.x;
  if (s >= ns) return;
  const bool bad = st->err_capacity != 0;
  if (bad || st->start_off[s] == st->start_off[s + 1]) o.hit_offset[(bad ? 0 : st->trk_off[s]) + s] = 0;
}

}  // namespace tpcca
