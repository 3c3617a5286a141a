// =========================================================================================
// tpcca_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded CPU statement of the five-stage cellular-automaton TPC
// sector tracker that BASELINE.json:5 (north_star) names and SURVEY.md section 8(c) /
// DESIGN.md section 3 define step by step.  The paper itself (section 1) only
// names the task ("full online track reconstruction of the TPC data ... the most
// computing-intense part of the synchronous processing"); it prints no algorithm and no
// numbers, so the result is a heuristic *defined by its algorithm* and this file follows
// that algorithm in DESIGN.md's order and notation, one IEEE operation per written
// operation, no blocking, no fusion, no reordering.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may load this library.  It shares no code, header, table generator or helper with the
// CUDA path (paper_2208_07412_b200/csrc); inputs and data tables come from tpcsynth/.
//
// Build: g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC  (see oracle/build.py).
//   Real = float  : the parity reference (north_star fixes fp32 arithmetic);
//   Real = double : same source, used only by the pins (P4, P6, P7).
//
// Pins (tests/test_oracle_pins.py): P1 grid invariants, P2 brute-force all-pairs neighbour
// search, P3 bin-size / mirror metamorphic, P4 exact straight-track recovery (dyadic
// geometry, score == 0), P5 link invariants, P6 noise-free helix recovery 1e-5 (double),
// P7 textbook weighted-least-squares reduction, P8 pulls / chi2, P9 covariance sanity,
// P10 generator truth (efficiency / fake), P11 determinism, P12 z-translation, plus a
// finite-difference pin of the transport Jacobian; the S5 DECISIONS (gap counting, phase-A
// gate, tc_min_hits, search window / tie-break, chi2 gate, readings R2 / R3) by the
// hand-worked toy tests/golden/toy_tracklets.txt and by the one-bin-per-row (brute-force
// search) metamorphic pin; tests/mutation_check.py re-checks that one-line mutations of
// those decisions fail a pin.  S6 / S7 / S8 (added in round 2 as new code below the five
// stages): hand-worked toys toy_selector.txt / toy_merge.txt, sort formulation, closed-form circle, exact circle
// geometry in two sector frames, finite-difference Jacobian of Rotate, generator truth.  Nothing can be pinned to
// values the paper prints (it prints none) -- "parity unpinned to the paper" in that sense only.
// =========================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

extern "C" {
struct oracle_params {      // all tables are double arrays holding the (fp32-representable) data
  int32_t n_rows;
  const double* row_x;
  const double* grid_y_lo;
  const double* grid_inv_bin_y;
  const int32_t* grid_ny;
  double grid_z_lo;
  const double* grid_inv_bin_z;
  const int32_t* grid_nz;
  const double* nf_hy_up;
  const double* nf_hz_up;
  const double* nf_hy_dn;
  const double* nf_hz_dn;
  const double* nf_cut;
  double kappa_per_qpt, err2_y, err2_z;
  double init_cov[5];
  double tc_win_y, tc_win_z, tc_gate, max_sinphi, grid_margin;
  int32_t tc_max_gap, tc_min_hits;
  int32_t sel_max_shared_permille;   // S6: a tracklet survives iff shared hits * 1000 <= this * n_hits
  double res_inv_quantum;            // S7: residuals are quantised to round(res * this), 16 bits
  // S8: cross-sector merging
  int32_t sectors_per_side;          // sectors s and s' are neighbours iff same side (s / this) and |s - s'| = 1 mod this
  double sector_cos, sector_sin;     // cos / sin of the angle between neighbouring sectors (20 degrees)
  int32_t mg_max_row_gap;            // the upper segment starts 1 .. this rows above the last row of the lower one
  double mg_dy, mg_dz, mg_dsin;      // match windows on y, z, sin(phi) at the upper segment's reference plane
  double mg_zpre;                    // pre-cut on |z(b at x_ref) - z(a on its last row)| before any transport
};
}

namespace {

constexpr int MAX_ROWS = 1024;

// lower-triangle index, i >= j
inline int tri(int i, int j) { return i * (i + 1) / 2 + j; }

template <class R>
struct KFState {
  R x;        // plane
  R p[5];     // y, z_rel, sin(phi), dz/ds, q/pT
  R C[15];    // lower triangle
  R chi2;
  int n;
  R c(int i, int j) const { return i >= j ? C[tri(i, j)] : C[tri(j, i)]; }
};

template <class R>
struct Track {
  R x_ref, z_ref, p[5], C[15], chi2;
  int32_t n_hits, n_fit, first_row, last_row, start_hit;
};

// ----------------------------------------------------------------------------- S6: tracklet selector
// SURVEY.md 8(f)-1 / DESIGN.md 3.7: "per-cluster ownership by (nHits, -trackId) ..., drop tracklets sharing
// more than X % of hits".  Integers only.  Tracks are numbered in output (start-hit) order.
//   owner[c]  = the track holding cluster c with the most hits; ties -> the smallest track number; -1 if none
//   n_own[t]  = hits of t that t owns;  shared(t) = n_hits(t) - n_own[t]
//   t is selected iff shared(t) * 1000 <= max_shared_permille * n_hits(t)
// (with four near-identical clones per long track -- reading N3 -- the longest clone owns everything
// the clones share and the others are dropped).
inline void select_tracks_plain(int64_t n_clusters, int64_t n_tracks, const int32_t* hit_offset, const int32_t* hit_idx,
                                int32_t max_shared_permille, std::vector<int32_t>& owner, std::vector<int32_t>& n_own,
                                std::vector<int32_t>& selected) {
  owner.assign(n_clusters, -1);
  n_own.assign(n_tracks, 0);
  selected.clear();
  for (int64_t t = 0; t < n_tracks; ++t) {
    const int32_t nh = hit_offset[t + 1] - hit_offset[t];
    for (int32_t k = hit_offset[t]; k < hit_offset[t + 1]; ++k) {
      const int32_t c = hit_idx[k];
      const int32_t o = owner[c];
      // t ascends, so on equal hit counts the earlier (smaller) track keeps the cluster
      if (o < 0 || nh > hit_offset[o + 1] - hit_offset[o]) owner[c] = (int32_t)t;
    }
  }
  for (int64_t t = 0; t < n_tracks; ++t)
    for (int32_t k = hit_offset[t]; k < hit_offset[t + 1]; ++k)
      if (owner[hit_idx[k]] == (int32_t)t) n_own[t]++;
  for (int64_t t = 0; t < n_tracks; ++t) {
    const int64_t nh = hit_offset[t + 1] - hit_offset[t];
    const int64_t shared = nh - n_own[t];
    if (shared * 1000 <= (int64_t)max_shared_permille * nh) selected.push_back((int32_t)t);
  }
}

template <class R>
class Oracle {
 public:
  explicit Oracle(const oracle_params& q) {
    n_rows = q.n_rows;
    auto cp = [&](std::vector<R>& v, const double* s) {
      v.resize(n_rows);
      for (int i = 0; i < n_rows; ++i) v[i] = (R)s[i];
    };
    cp(row_x, q.row_x); cp(grid_y_lo, q.grid_y_lo); cp(inv_bin_y, q.grid_inv_bin_y);
    cp(inv_bin_z, q.grid_inv_bin_z); cp(hy_up, q.nf_hy_up); cp(hz_up, q.nf_hz_up);
    cp(hy_dn, q.nf_hy_dn); cp(hz_dn, q.nf_hz_dn); cp(nf_cut, q.nf_cut);
    ny.assign(q.grid_ny, q.grid_ny + n_rows);
    nz.assign(q.grid_nz, q.grid_nz + n_rows);
    grid_z_lo = (R)q.grid_z_lo;
    Bc = (R)q.kappa_per_qpt; err2_y = (R)q.err2_y; err2_z = (R)q.err2_z;
    for (int i = 0; i < 5; ++i) init_cov[i] = (R)q.init_cov[i];
    win_y = (R)q.tc_win_y; win_z = (R)q.tc_win_z; gate = (R)q.tc_gate;
    max_sinphi = (R)q.max_sinphi; margin = (R)q.grid_margin;
    max_gap = q.tc_max_gap; min_hits = q.tc_min_hits;
    sel_permille = q.sel_max_shared_permille;
    res_inv_q = (R)q.res_inv_quantum;
    per_side = q.sectors_per_side; sec_cos = (R)q.sector_cos; sec_sin = (R)q.sector_sin;
    mg_gap = q.mg_max_row_gap; mg_dy = (R)q.mg_dy; mg_dz = (R)q.mg_dz; mg_ds = (R)q.mg_dsin; mg_zpre = (R)q.mg_zpre;
    row_bin_base.resize(n_rows + 1);
    row_bin_base[0] = 0;
    for (int r = 0; r < n_rows; ++r) row_bin_base[r + 1] = row_bin_base[r] + (int64_t)ny[r] * nz[r];
    c24 = (R)(1.0 / 24.0); c640 = (R)(3.0 / 640.0); c12 = (R)(1.0 / 12.0);
  }

  // ----------------------------------------------------------------------------- S1
  // by = clamp(floor((y - grid_y_lo_r) * inv_bin_y_r), 0, ny_r - 1), same for
  // z; bin = bz * ny_r + by (y fastest).
  int bin_y(int r, R y) const {
    R t = (y - grid_y_lo[r]) * inv_bin_y[r];
    R f = std::floor(t);
    if (f < (R)0) f = (R)0;
    R hi = (R)(ny[r] - 1);
    if (f > hi) f = hi;
    return (int)f;
  }
  int bin_z(int r, R z) const {
    R t = (z - grid_z_lo) * inv_bin_z[r];
    R f = std::floor(t);
    if (f < (R)0) f = (R)0;
    R hi = (R)(nz[r] - 1);
    if (f > hi) f = hi;
    return (int)f;
  }

  int load(int64_t n_, const R* y_, const R* z_, const uint16_t* row_) {
    n = n_;
    for (int64_t i = 0; i < n; ++i)
      if (row_[i] >= n_rows) return -5;
    y.assign(y_, y_ + n); z.assign(z_, z_ + n); row.assign(row_, row_ + n);
    return 0;
  }

  // sorted order = ascending (row, bin, original index); bin_start = exclusive prefix of the
  // per-bin counts (sector-local sorted positions), row_start[r] = first position of row r.
  void build_grid() {
    std::vector<uint64_t> key(n);      // global bin id of the sector
    for (int64_t i = 0; i < n; ++i) {
      int r = row[i];
      int by = bin_y(r, y[i]);
      int bz = bin_z(r, z[i]);
      key[i] = (uint64_t)(row_bin_base[r] + (int64_t)bz * ny[r] + by);
    }
    order.resize(n);
    for (int64_t i = 0; i < n; ++i) order[i] = (int32_t)i;
    std::sort(order.begin(), order.end(), [&](int32_t a, int32_t b) {
      if (key[a] != key[b]) return key[a] < key[b];
      return a < b;
    });
    int64_t nb = row_bin_base[n_rows];
    bin_start.assign(nb + 1, 0);
    for (int64_t i = 0; i < n; ++i) bin_start[key[i] + 1]++;
    for (int64_t b = 0; b < nb; ++b) bin_start[b + 1] += bin_start[b];
    sy.resize(n); sz.resize(n); srow.resize(n);
    for (int64_t p = 0; p < n; ++p) {
      sy[p] = y[order[p]]; sz[p] = z[order[p]]; srow[p] = row[order[p]];
    }
    row_start.assign(n_rows + 1, 0);
    for (int r = 0; r <= n_rows; ++r) row_start[r] = (int32_t)bin_start[row_bin_base[r]];
  }

  // ----------------------------------------------------------------------------- S2
  // candidates of row r2 inside the window |y - yc| <= hy and |z - zc| <= hz; brute = whole row
  void window(int r2, R yc, R zc, R hy, R hz, bool brute, std::vector<int32_t>& out) const {
    out.clear();
    if (brute) {
      for (int32_t c = row_start[r2]; c < row_start[r2 + 1]; ++c) {
        R dy = sy[c] - yc, dz = sz[c] - zc;
        if (std::fabs(dy) <= hy && std::fabs(dz) <= hz) out.push_back(c);
      }
      return;
    }
    // the grid is only an accelerator: visit a superset of the window, then the exact test
    R my = hy + margin, mz = hz + margin;
    int by0 = bin_y(r2, yc - my), by1 = bin_y(r2, yc + my);
    int bz0 = bin_z(r2, zc - mz), bz1 = bin_z(r2, zc + mz);
    for (int bz = bz0; bz <= bz1; ++bz) {
      int64_t b0 = row_bin_base[r2] + (int64_t)bz * ny[r2];
      for (uint32_t c = bin_start[b0 + by0]; c < bin_start[b0 + by1 + 1]; ++c) {
        R dy = sy[c] - yc, dz = sz[c] - zc;
        if (std::fabs(dy) <= hy && std::fabs(dz) <= hz) out.push_back((int32_t)c);
      }
    }
  }

  // score of the triplet (d, c, u)
  R score(int r, R yc, R zc, R yu, R zu, R yd, R zd) const {
    R dxu = row_x[r + 1] - row_x[r];
    R dxd = row_x[r] - row_x[r - 1];
    R ay = (yu - yc) * dxd - (yc - yd) * dxu;
    R az = (zu - zc) * dxd - (zc - zd) * dxu;
    return ay * ay + az * az;
  }

  void find_neighbours(bool brute) {
    link_up.assign(n, -1); link_dn.assign(n, -1);
    std::vector<int32_t> U, D;
    for (int64_t c = 0; c < n; ++c) {
      int r = srow[c];
      if (r < 1 || r > n_rows - 2) continue;
      R yc = sy[c], zc = sz[c];
      window(r + 1, yc, zc, hy_up[r], hz_up[r], brute, U);
      if (U.empty()) continue;
      window(r - 1, yc, zc, hy_dn[r], hz_dn[r], brute, D);
      if (D.empty()) continue;
      bool have = false;
      R best = 0; int32_t bu = -1, bd = -1;
      for (int32_t u : U)
        for (int32_t d : D) {
          R s = score(r, yc, zc, sy[u], sz[u], sy[d], sz[d]);
          bool better;
          if (!have) better = true;
          else if (s < best) better = true;
          else if (s == best) {
            // ties: smallest original id of u, then of d
            if (order[u] != order[bu]) better = order[u] < order[bu];
            else better = order[d] < order[bd];
          } else better = false;
          if (better) { have = true; best = s; bu = u; bd = d; }
        }
      if (have && best <= nf_cut[r]) { link_up[c] = bu; link_dn[c] = bd; }
    }
  }

  // ----------------------------------------------------------------------------- S3 / S4
  void clean_links() {
    link_up_c.assign(n, -1); link_dn_c.assign(n, -1);
    for (int64_t c = 0; c < n; ++c) {
      int32_t u = link_up[c], d = link_dn[c];
      if (u >= 0 && link_dn[u] == (int32_t)c) link_up_c[c] = u;
      if (d >= 0 && link_up[d] == (int32_t)c) link_dn_c[c] = d;
    }
  }
  void select_start_hits() {
    start_hit.clear();
    for (int64_t c = 0; c < n; ++c)
      if (link_dn_c[c] == -1 && link_up_c[c] >= 0) start_hit.push_back((int32_t)c);
  }

  // ----------------------------------------------------------------------------- S5: Kalman
  // DESIGN.md 3.5 "Propagate to x2".  Returns false (state untouched) on failure.
  bool propagate(KFState<R>& s, R x2) const {
    R dx = x2 - s.x;
    if (dx == (R)0) return true;
    R k = s.p[4] * Bc;
    R ey = s.p[2];
    R ey2 = ey + k * dx;
    if (!(std::fabs(ey) <= max_sinphi) || !(std::fabs(ey2) <= max_sinphi)) return false;
    R ex = std::sqrt((R)1 - ey * ey);
    R ex2 = std::sqrt((R)1 - ey2 * ey2);
    R sx = ex + ex2;
    R sY = ey + ey2;
    R tg = sY / sx;
    R dy = dx * tg;
    R d2 = dx * dx + dy * dy;
    R d = std::sqrt(d2);
    if (dx < (R)0) d = -d;
    R tt = (k * k) * d2;
    R dS = d * ((R)1 + tt * (c24 + tt * c640));
    R cc = (R)1 + (ex * ex2 + ey * ey2);
    R n02 = (dx * cc) / ((sx * ex) * ex2);
    R j4 = ((dx * dx) * cc) / (ex2 * (sx * sx));
    R n04 = Bc * j4;
    R n12 = s.p[3] * ((dx * tg) / (ex * ex2));
    R n13 = dS;
    R n14 = (s.p[3] * Bc) * ((dy / d) * j4 + ((k * d) * d2) * c12);
    R n24 = Bc * dx;
    s.p[0] = s.p[0] + dy;
    s.p[1] = s.p[1] + s.p[3] * dS;
    s.p[2] = ey2;
    s.x = x2;
    // A = J*C (all 25), then C' = A*J^T (lower triangle); terms added left to right
    R A[5][5];
    for (int j = 0; j < 5; ++j) {
      A[0][j] = s.c(0, j) + n02 * s.c(2, j) + n04 * s.c(4, j);
      A[1][j] = s.c(1, j) + n12 * s.c(2, j) + n13 * s.c(3, j) + n14 * s.c(4, j);
      A[2][j] = s.c(2, j) + n24 * s.c(4, j);
      A[3][j] = s.c(3, j);
      A[4][j] = s.c(4, j);
    }
    for (int i = 0; i < 5; ++i) {
      s.C[tri(i, 0)] = A[i][0] + A[i][2] * n02 + A[i][4] * n04;
      if (i >= 1) s.C[tri(i, 1)] = A[i][1] + A[i][2] * n12 + A[i][3] * n13 + A[i][4] * n14;
      if (i >= 2) s.C[tri(i, 2)] = A[i][2] + A[i][4] * n24;
      if (i >= 3) s.C[tri(i, 3)] = A[i][3];
      if (i >= 4) s.C[tri(i, 4)] = A[i][4];
    }
    return true;
  }

  // gate distance on the predicted state
  R dist2(const KFState<R>& s, R ym, R zm) const {
    R ry = ym - s.p[0];
    R rz = zm - s.p[1];
    return (ry * ry) / (s.C[tri(0, 0)] + err2_y) + (rz * rz) / (s.C[tri(1, 1)] + err2_z);
  }

  // one scalar update of component m (0 = y, 1 = z) with variance e2
  void update1(KFState<R>& s, int m, R meas, R e2) const {
    R r = meas - s.p[m];
    R w = (R)1 / (s.C[tri(m, m)] + e2);
    R col[5], kk[5];
    for (int i = 0; i < 5; ++i) col[i] = s.c(i, m);
    for (int i = 0; i < 5; ++i) { kk[i] = col[i] * w; s.p[i] = s.p[i] + kk[i] * r; }
    for (int i = 0; i < 5; ++i)
      for (int j = 0; j <= i; ++j) s.C[tri(i, j)] = s.C[tri(i, j)] - kk[i] * col[j];
    s.chi2 = s.chi2 + (r * r) * w;
  }
  void update(KFState<R>& s, R ym, R zm) const {
    update1(s, 0, ym, err2_y);
    update1(s, 1, zm, err2_z);
    s.n++;
  }

  // Search(row r): best cluster inside the tc window around the prediction; ties -> smallest id
  int32_t search(const KFState<R>& s, int r, R z_ref, R& best_d2) const {
    R yc = s.p[0];
    R zc = z_ref + s.p[1];
    R my = win_y + margin, mz = win_z + margin;
    int by0 = bin_y(r, yc - my), by1 = bin_y(r, yc + my);
    int bz0 = bin_z(r, zc - mz), bz1 = bin_z(r, zc + mz);
    R wy = s.C[tri(0, 0)] + err2_y;
    R wz = s.C[tri(1, 1)] + err2_z;
    int32_t best = -1;
    for (int bz = bz0; bz <= bz1; ++bz) {
      int64_t b0 = row_bin_base[r] + (int64_t)bz * ny[r];
      for (uint32_t c = bin_start[b0 + by0]; c < bin_start[b0 + by1 + 1]; ++c) {
        R ry = sy[c] - s.p[0];
        R rz = (sz[c] - z_ref) - s.p[1];
        if (!(std::fabs(ry) <= win_y && std::fabs(rz) <= win_z)) continue;
        R d2 = (ry * ry) / wy + (rz * rz) / wz;
        if (best < 0 || d2 < best_d2 || (d2 == best_d2 && order[c] < order[best])) {
          best = (int32_t)c; best_d2 = d2;
        }
      }
    }
    return best;
  }

  void reset_cov(KFState<R>& s) const {
    for (int i = 0; i < 15; ++i) s.C[i] = (R)0;
    for (int i = 0; i < 5; ++i) s.C[tri(i, i)] = init_cov[i];
    s.chi2 = (R)0;
    s.n = 0;
  }

  // seed, phase A (follow links), phase B (extrapolate up), phase C (refit down)
  bool construct_tracklet(int32_t c0, Track<R>& out, std::vector<int32_t>& hit) const {
    int r0 = srow[c0];
    int32_t c1 = link_up_c[c0];
    R z_ref = sz[c0];
    KFState<R> s;
    {
      R dx = row_x[r0 + 1] - row_x[r0];
      R dy = sy[c1] - sy[c0];
      R dz = sz[c1] - z_ref;
      R d = std::sqrt(dx * dx + dy * dy);
      s.x = row_x[r0];
      s.p[0] = sy[c0]; s.p[1] = (R)0; s.p[2] = dy / d; s.p[3] = dz / d; s.p[4] = (R)0;
      reset_cov(s);
    }
    hit.assign(n_rows, -1);
    int top = r0;
    bool failed = false;
    // ---- phase A
    int32_t cur = c0;
    int last = r0;
    while (cur != -1) {
      int r = srow[cur];
      if (!propagate(s, row_x[r])) { failed = true; break; }
      R ym = sy[cur], zm = sz[cur] - z_ref;
      if (s.n >= 2 && dist2(s, ym, zm) > gate) break;
      update(s, ym, zm);
      hit[r] = cur; last = r; top = r;
      cur = link_up_c[cur];
    }
    // ---- phase B
    if (!failed) {
      int gap = 0;
      for (int r = last + 1; r < n_rows; ++r) {
        if (!propagate(s, row_x[r])) break;
        R d2 = (R)0;
        int32_t b = search(s, r, z_ref, d2);
        if (b >= 0 && d2 <= gate) {
          update(s, sy[b], sz[b] - z_ref);
          hit[r] = b; top = r; gap = 0;
        } else {
          if (++gap > max_gap) break;
        }
      }
    }
    // ---- phase C: start at the highest row holding a hit (DESIGN.md 3.8 reading R2)
    reset_cov(s);
    int gap = 0;
    bool have_snap = false;
    KFState<R> snap = s;
    for (int r = top; r >= 0; --r) {
      if (!propagate(s, row_x[r])) break;
      if (hit[r] != -1) {
        int32_t c = hit[r];
        update(s, sy[c], sz[c] - z_ref);
        snap = s; have_snap = true;
      } else {
        bool took = false;
        if (s.n >= 2) {   // reading R3: no search before two hits constrain the direction
          R d2 = (R)0;
          int32_t b = search(s, r, z_ref, d2);
          if (b >= 0 && d2 <= gate) {
            update(s, sy[b], sz[b] - z_ref);
            hit[r] = b; snap = s; have_snap = true; gap = 0; took = true;
          }
        }
        if (!took && r < r0) {
          if (++gap > max_gap) break;
        }
      }
    }
    int nh = 0, first = -1, lastr = -1;
    for (int r = 0; r < n_rows; ++r)
      if (hit[r] != -1) { if (first < 0) first = r; lastr = r; ++nh; }
    if (nh < min_hits || !have_snap) return false;
    out.x_ref = snap.x; out.z_ref = z_ref;
    for (int i = 0; i < 5; ++i) out.p[i] = snap.p[i];
    for (int i = 0; i < 15; ++i) out.C[i] = snap.C[i];
    out.chi2 = snap.chi2; out.n_fit = snap.n; out.n_hits = nh;
    out.first_row = first; out.last_row = lastr; out.start_hit = c0;
    return true;
  }

  void construct_tracklets() {
    tracks.clear(); hit_offset.assign(1, 0); hit_idx.clear();
    std::vector<int32_t> hit;
    for (int32_t c0 : start_hit) {
      Track<R> t;
      if (!construct_tracklet(c0, t, hit)) continue;
      tracks.push_back(t);
      for (int r = 0; r < n_rows; ++r)
        if (hit[r] != -1) hit_idx.push_back(hit[r]);
      hit_offset.push_back((int32_t)hit_idx.size());
    }
  }

  // ----------------------------------------------------------------------------- S7: track residuals
  // SURVEY.md 8(f)-4 / DESIGN.md 3.7: the front end of a track-model cluster compression ("data
  // compression rely on the information from TPC tracking").  For every SELECTED track t (S6), starting from its
  // fitted state (x_ref, p) and walking its hits in ascending row, the state is transported hit to hit with
  // Propagate (mean only: the covariance is not needed) and, for every hit c that t OWNS,
  //   res_y[c] = y_c - p0,   res_z[c] = (z_c - z_ref) - p1,   q_y = clamp(rint(res_y * inv_quantum), +-32767), q_z likewise
  // (rint = round half to even, the fp32 decision), res_trk[c] = t.  A failed transport ends the track's walk.
  // Clusters no selected track owns keep res_trk = -1, residuals 0 (a codec stores them raw).
  void track_residuals() {
    res_trk.assign(n, -1); res_y.assign(n, (R)0); res_z.assign(n, (R)0); q_y.assign(n, 0); q_z.assign(n, 0);
    out_state.assign(selected.size(), KFState<R>());
    out_ok.assign(selected.size(), 0);
    size_t ksel = 0;
    for (int32_t t : selected) {
      const Track<R>& T = tracks[t];
      KFState<R> s;
      s.x = T.x_ref;
      for (int i = 0; i < 5; ++i) s.p[i] = T.p[i];
      for (int i = 0; i < 15; ++i) s.C[i] = (R)0;
      s.chi2 = (R)0; s.n = 0;
      bool walked = true;
      for (int32_t k = hit_offset[t]; k < hit_offset[t + 1]; ++k) {
        const int32_t c = hit_idx[k];
        if (!propagate(s, row_x[srow[c]])) { walked = false; break; }
        if (k + 1 == hit_offset[t + 1]) { out_state[ksel] = s; out_ok[ksel] = 1; }   // S8: state on the last row
        if (owner[c] != t) continue;
        const R ry = sy[c] - s.p[0];
        const R rz = (sz[c] - T.z_ref) - s.p[1];
        res_trk[c] = t; res_y[c] = ry; res_z[c] = rz;
        q_y[c] = quantise(ry); q_z[c] = quantise(rz);
      }
      (void)walked;
      ++ksel;
    }
  }
  int16_t quantise(R r) const {
    R v = std::nearbyint(r * res_inv_q);          // default rounding mode: half to even
    if (v > (R)32767) v = (R)32767;
    if (v < (R)-32767) v = (R)-32767;
    return (int16_t)v;
  }

  // ----------------------------------------------------------------------------- S8: cross-sector merging
  // DESIGN.md 3.7 "Rotate": the state at plane x of a frame is re-expressed in the frame turned by the angle
  // whose cosine / sine are (ca, sa) (sa > 0: towards the next sector in azimuth), at the plane through the SAME
  // space point:  x' = x ca + y sa,  y' = y ca - x sa,  sin phi' = sin phi ca - cos phi sa  (cos phi > 0: the
  // track moves outward).  Covariance: a shift dy of the point moves it by (dy sa, dy ca) in the new frame; back
  // on the fixed plane x' that is  dY = dy cos phi / cos phi',  dZ = -dy p3 sa / cos phi',
  // d sin phi' = -dy (Bc p4) sa;  and  d sin phi' / d sin phi = cos phi' / cos phi.  Fails (state untouched) if
  // |sin phi| or |sin phi'| exceeds max_sinphi.
  bool rotate(KFState<R>& s, R ca, R sa) const {
    const R sf = s.p[2];
    if (!(std::fabs(sf) <= max_sinphi)) return false;
    const R cf = std::sqrt((R)1 - sf * sf);
    const R sf2 = sf * ca - cf * sa;
    if (!(std::fabs(sf2) <= max_sinphi)) return false;
    const R cf2 = std::sqrt((R)1 - sf2 * sf2);
    const R x2 = s.x * ca + s.p[0] * sa;
    const R y2 = s.p[0] * ca - s.x * sa;
    const R j00 = cf / cf2;
    const R j10 = -((s.p[3] * sa) / cf2);
    const R j20 = -((s.p[4] * Bc) * sa);
    const R j22 = cf2 / cf;
    R A[5][5];
    for (int j = 0; j < 5; ++j) {
      A[0][j] = j00 * s.c(0, j);
      A[1][j] = j10 * s.c(0, j) + s.c(1, j);
      A[2][j] = j20 * s.c(0, j) + j22 * s.c(2, j);
      A[3][j] = s.c(3, j);
      A[4][j] = s.c(4, j);
    }
    for (int i = 0; i < 5; ++i) {
      s.C[tri(i, 0)] = A[i][0] * j00;
      if (i >= 1) s.C[tri(i, 1)] = A[i][0] * j10 + A[i][1];
      if (i >= 2) s.C[tri(i, 2)] = A[i][0] * j20 + A[i][2] * j22;
      if (i >= 3) s.C[tri(i, 3)] = A[i][3];
      if (i >= 4) s.C[tri(i, 4)] = A[i][4];
    }
    s.x = x2; s.p[0] = y2; s.p[2] = sf2;
    return true;
  }

  void run(uint32_t stage_mask, bool brute) {
    if (stage_mask & 1u) build_grid();
    if (stage_mask & 2u) find_neighbours(brute);
    if (stage_mask & 4u) clean_links();
    if (stage_mask & 8u) select_start_hits();
    if (stage_mask & 16u) construct_tracklets();
    if (stage_mask & 32u)
      select_tracks_plain(n, (int64_t)tracks.size(), hit_offset.data(), hit_idx.data(), sel_permille, owner, n_own, selected);
    if (stage_mask & 64u) track_residuals();
  }

  // tables
  int n_rows;
  std::vector<R> row_x, grid_y_lo, inv_bin_y, inv_bin_z, hy_up, hz_up, hy_dn, hz_dn, nf_cut;
  std::vector<int32_t> ny, nz;
  std::vector<int64_t> row_bin_base;
  R grid_z_lo, Bc, err2_y, err2_z, init_cov[5], win_y, win_z, gate, max_sinphi, margin;
  R c24, c640, c12;
  int max_gap, min_hits, sel_permille;
  R res_inv_q;
  int per_side = 0, mg_gap = 0;
  R sec_cos = 0, sec_sin = 0, mg_dy = 0, mg_dz = 0, mg_ds = 0, mg_zpre = 0;
  // data
  int64_t n = 0;
  std::vector<R> y, z, sy, sz;
  std::vector<uint16_t> row, srow;
  std::vector<int32_t> order, row_start;
  std::vector<uint32_t> bin_start;
  std::vector<int32_t> link_up, link_dn, link_up_c, link_dn_c, start_hit;
  std::vector<Track<R>> tracks;
  std::vector<int32_t> hit_offset, hit_idx;
  std::vector<int32_t> owner, n_own, selected;   // S6
  std::vector<int32_t> res_trk;                  // S7
  std::vector<R> res_y, res_z;
  std::vector<int16_t> q_y, q_z;
  std::vector<KFState<R>> out_state;             // S7 by-product for S8: state of each selected track on its last row
  std::vector<char> out_ok;
  // S8, per selected track: neighbour-sector partner above (next) / below (prev), -1 none
  std::vector<int32_t> mg_next_sec, mg_next_trk, mg_prev_sec, mg_prev_trk;
  struct Merged { int32_t head; std::vector<int32_t> seg_sec, seg_trk; Track<R> t; };
  std::vector<Merged> merged;                     // chains whose lowest segment lives in this sector
};

// S8: match the selected tracks of neighbouring sectors and refit the chains.
//  Matching.  a = selected track of sector s with an outer state (S7 walk), b = selected track of a neighbour
//  sector n (same side, next or previous in azimuth) with 1 <= first_row(b) - last_row(a) <= mg_max_row_gap and
//  |(z_ref(b) + p1(b)) - (z_ref(a) + p1_out(a))| <= mg_zpre (a cheap pre-cut an index can serve):
//  a's outer state is rotated into n's frame and propagated to x_ref(b) (either failing: no candidate), then
//    dy = p0(b) - p0',  dz = (z_ref(b) - z_ref(a)) + (p1(b) - p1'),  ds = p2(b) - p2';
//  candidate iff |dy| <= mg_dy, |dz| <= mg_dz, |ds| <= mg_dsin;  score = (dy/mg_dy)^2 + (dz/mg_dz)^2 + (ds/mg_dsin)^2.
//  next(a) = the candidate with the smallest score (ties: smaller sector, then smaller track), prev(b) likewise
//  over the a's that have b as a candidate; the link a -> b is kept iff next(a) = b and prev(b) = a.
//  Refit.  For every chain g1 -> ... -> gk (g1 has no prev): start from gk's outer state with the reset
//  covariance and run the Kalman filter downward over the hits of gk, ..., g1 (propagate to the hit's row,
//  update; no gate, no search); between segments the state is rotated into the lower segment's frame and p1 is
//  re-referenced: p1 += z_ref(upper) - z_ref(lower).  A failed transport / rotation ends the refit (the chain
//  is emitted with what was fitted if at least one update happened).
template <class R>
void merge_sectors(std::vector<Oracle<R>*>& S) {
  const int ns = (int)S.size();
  for (auto* o : S) {
    const size_t k = o->selected.size();
    o->mg_next_sec.assign(k, -1); o->mg_next_trk.assign(k, -1); o->mg_prev_sec.assign(k, -1); o->mg_prev_trk.assign(k, -1);
    o->merged.clear();
  }
  if (ns == 0) return;
  const int per = S[0]->per_side;
  if (per < 2 || ns % per != 0) return;                 // no neighbour relation defined
  struct Best { bool have = false; R score = 0; int sec = -1, trk = -1; };
  std::vector<std::vector<Best>> nxt(ns), prv(ns);
  for (int s = 0; s < ns; ++s) { nxt[s].assign(S[s]->selected.size(), Best()); prv[s].assign(S[s]->selected.size(), Best()); }
  auto better = [](const Best& b, R sc, int sec, int trk) {
    if (!b.have) return true;
    if (sc != b.score) return sc < b.score;
    if (sec != b.sec) return sec < b.sec;
    return trk < b.trk;
  };
  for (int s = 0; s < ns; ++s) {
    Oracle<R>& A = *S[s];
    const int side = s / per, loc = s % per;
    for (int dir = 0; dir < 2; ++dir) {
      const int nsec = side * per + (dir == 0 ? (loc + 1) % per : (loc + per - 1) % per);
      if (nsec == s) continue;
      if (per == 2 && dir == 1) continue;               // two sectors per side: one neighbour, reached once
      Oracle<R>& B = *S[nsec];
      const R sa = dir == 0 ? A.sec_sin : -A.sec_sin;
      for (size_t ia = 0; ia < A.selected.size(); ++ia) {
        if (!A.out_ok[ia]) continue;
        const Track<R>& ta = A.tracks[A.selected[ia]];
        for (size_t ib = 0; ib < B.selected.size(); ++ib) {
          const Track<R>& tb = B.tracks[B.selected[ib]];
          const int gap = tb.first_row - ta.last_row;
          if (gap < 1 || gap > A.mg_gap) continue;
          const R za = ta.z_ref + A.out_state[ia].p[1], zb = tb.z_ref + tb.p[1];
          if (!(std::fabs(zb - za) <= A.mg_zpre)) continue;
          KFState<R> st = A.out_state[ia];
          if (!A.rotate(st, A.sec_cos, sa)) continue;
          if (!A.propagate(st, tb.x_ref)) continue;
          const R dy = tb.p[0] - st.p[0];
          const R dz = (tb.z_ref - ta.z_ref) + (tb.p[1] - st.p[1]);
          const R ds = tb.p[2] - st.p[2];
          if (!(std::fabs(dy) <= A.mg_dy && std::fabs(dz) <= A.mg_dz && std::fabs(ds) <= A.mg_ds)) continue;
          const R qy = dy / A.mg_dy, qz = dz / A.mg_dz, qs = ds / A.mg_ds;
          const R sc = qy * qy + qz * qz + qs * qs;
          if (better(nxt[s][ia], sc, nsec, (int)ib)) { nxt[s][ia].have = true; nxt[s][ia].score = sc; nxt[s][ia].sec = nsec; nxt[s][ia].trk = (int)ib; }
          if (better(prv[nsec][ib], sc, s, (int)ia)) { prv[nsec][ib].have = true; prv[nsec][ib].score = sc; prv[nsec][ib].sec = s; prv[nsec][ib].trk = (int)ia; }
        }
      }
    }
  }
  for (int s = 0; s < ns; ++s)
    for (size_t ia = 0; ia < S[s]->selected.size(); ++ia) {
      const Best& b = nxt[s][ia];
      if (!b.have) continue;
      const Best& back = prv[b.sec][b.trk];
      if (back.have && back.sec == s && back.trk == (int)ia) {
        S[s]->mg_next_sec[ia] = b.sec; S[s]->mg_next_trk[ia] = b.trk;
        S[b.sec]->mg_prev_sec[b.trk] = s; S[b.sec]->mg_prev_trk[b.trk] = (int32_t)ia;
      }
    }
  // ---- refit of the chains
  for (int s = 0; s < ns; ++s) {
    Oracle<R>& H = *S[s];
    for (size_t ih = 0; ih < H.selected.size(); ++ih) {
      if (H.mg_prev_sec[ih] != -1 || H.mg_next_sec[ih] == -1) continue;       // heads of chains with >= 2 segments
      typename Oracle<R>::Merged M;
      M.head = (int32_t)ih;
      int cs = s, ct = (int)ih;
      while (cs != -1) {
        M.seg_sec.push_back(cs); M.seg_trk.push_back(ct);
        const int ns2 = S[cs]->mg_next_sec[ct], nt2 = S[cs]->mg_next_trk[ct];
        cs = ns2; ct = nt2;
      }
      const int k = (int)M.seg_sec.size();
      Oracle<R>& Top = *S[M.seg_sec[k - 1]];
      KFState<R> st = Top.out_state[M.seg_trk[k - 1]];       // exists: the top segment was matched through it or ...
      bool ok = Top.out_ok[M.seg_trk[k - 1]] != 0;
      H.reset_cov(st);
      KFState<R> snap = st;
      bool have_snap = false;
      int n_hits = 0, first = -1, last = -1, g_snap = k - 1;
      for (int g = k - 1; g >= 0 && ok; --g) {
        Oracle<R>& G = *S[M.seg_sec[g]];
        const int32_t t = G.selected[M.seg_trk[g]];
        const Track<R>& tg = G.tracks[t];
        if (g < k - 1) {
          // into the lower segment's frame: the inverse of the rotation that led from it to the upper one
          const int up = M.seg_sec[g + 1], lo = M.seg_sec[g];
          const int per_ = G.per_side;
          const bool up_is_next = (up % per_) == ((lo % per_) + 1) % per_;
          const R sa = up_is_next ? -G.sec_sin : G.sec_sin;
          if (!G.rotate(st, G.sec_cos, sa)) { ok = false; break; }
          const Track<R>& tu = S[up]->tracks[S[up]->selected[M.seg_trk[g + 1]]];
          st.p[1] = st.p[1] + (tu.z_ref - tg.z_ref);
        }
        for (int32_t q = G.hit_offset[t + 1] - 1; q >= G.hit_offset[t]; --q) {
          const int32_t c = G.hit_idx[q];
          if (!G.propagate(st, G.row_x[G.srow[c]])) { ok = false; break; }
          G.update(st, G.sy[c], G.sz[c] - tg.z_ref);
          snap = st; have_snap = true; g_snap = g;
          if (last < 0) last = G.srow[c];
          first = G.srow[c];
          ++n_hits;
        }
      }
      if (!have_snap) continue;
      M.t.x_ref = snap.x;
      {   // the parameters are in the frame (and relative to the z_ref) of the lowest segment the refit reached
        Oracle<R>& G = *S[M.seg_sec[g_snap]];
        M.t.z_ref = G.tracks[G.selected[M.seg_trk[g_snap]]].z_ref;
        M.t.start_hit = g_snap;                     // index of that segment in the chain (0 = head: the normal case)
      }
      for (int i = 0; i < 5; ++i) M.t.p[i] = snap.p[i];
      for (int i = 0; i < 15; ++i) M.t.C[i] = snap.C[i];
      M.t.chi2 = snap.chi2; M.t.n_fit = snap.n; M.t.n_hits = n_hits; M.t.first_row = first; M.t.last_row = last;
      H.merged.push_back(M);
    }
  }
}

struct Handle {
  int precision;           // 0 = float, 1 = double
  Oracle<float>* f = nullptr;
  Oracle<double>* d = nullptr;
};

template <class V>
void copy_out(double* dst, const V& v) { for (size_t i = 0; i < v.size(); ++i) dst[i] = (double)v[i]; }

// state = [x, p0..p4, C0..C14, chi2] (22 doubles), in/out
template <class R>
void st_in(KFState<R>& s, const double* st) {
  s.x = (R)st[0];
  for (int i = 0; i < 5; ++i) s.p[i] = (R)st[1 + i];
  for (int i = 0; i < 15; ++i) s.C[i] = (R)st[6 + i];
  s.chi2 = (R)st[21]; s.n = 0;
}
template <class R>
void st_out(const KFState<R>& s, double* st) {
  st[0] = (double)s.x;
  for (int i = 0; i < 5; ++i) st[1 + i] = (double)s.p[i];
  for (int i = 0; i < 15; ++i) st[6 + i] = (double)s.C[i];
  st[21] = (double)s.chi2;
}

}  // namespace

#define DISPATCH(h, expr_f, expr_d) (((Handle*)(h))->precision == 0 ? (expr_f) : (expr_d))

extern "C" {

void* oracle_create(const oracle_params* q, int precision) {
  if (!q || q->n_rows < 3 || q->n_rows > MAX_ROWS) return nullptr;
  Handle* h = new Handle;
  h->precision = precision;
  if (precision == 0) h->f = new Oracle<float>(*q); else h->d = new Oracle<double>(*q);
  return h;
}
void oracle_destroy(void* hv) {
  Handle* h = (Handle*)hv;
  if (!h) return;
  delete h->f; delete h->d; delete h;
}
// y, z: float* if precision 0, double* if precision 1.  One sector.
int oracle_load(void* hv, int64_t n, const void* y, const void* z, const uint16_t* row) {
  Handle* h = (Handle*)hv;
  if (h->precision == 0) return h->f->load(n, (const float*)y, (const float*)z, row);
  return h->d->load(n, (const double*)y, (const double*)z, row);
}
// stage_mask bit i = stage i+1; brute != 0: S2 scans whole rows r+-1 instead of the grid
int oracle_run(void* hv, uint32_t stage_mask, int brute) {
  Handle* h = (Handle*)hv;
  if (h->precision == 0) h->f->run(stage_mask, brute != 0); else h->d->run(stage_mask, brute != 0);
  return 0;
}
// out[0..4] = n_clusters, n_start, n_tracks, n_hits, n_bins
void oracle_sizes(void* hv, int64_t* out) {
  Handle* h = (Handle*)hv;
#define SZ(o) do { out[0] = (o)->n; out[1] = (int64_t)(o)->start_hit.size(); \
    out[2] = (int64_t)(o)->tracks.size(); out[3] = (int64_t)(o)->hit_idx.size(); \
    out[4] = (o)->row_bin_base[(o)->n_rows]; } while (0)
  if (h->precision == 0) SZ(h->f); else SZ(h->d);
#undef SZ
}
void oracle_get_grid(void* hv, int32_t* order, double* sy, double* sz, uint32_t* bin_start, int32_t* row_start) {
  Handle* h = (Handle*)hv;
#define GG(o) do { \
    if (order) std::copy((o)->order.begin(), (o)->order.end(), order); \
    if (sy) copy_out(sy, (o)->sy); \
    if (sz) copy_out(sz, (o)->sz); \
    if (bin_start) std::copy((o)->bin_start.begin(), (o)->bin_start.end(), bin_start); \
    if (row_start) std::copy((o)->row_start.begin(), (o)->row_start.end(), row_start); } while (0)
  if (h->precision == 0) GG(h->f); else GG(h->d);
#undef GG
}
void oracle_get_links(void* hv, int32_t* up_raw, int32_t* dn_raw, int32_t* up, int32_t* dn, int32_t* start) {
  Handle* h = (Handle*)hv;
#define GL(o) do { \
    if (up_raw) std::copy((o)->link_up.begin(), (o)->link_up.end(), up_raw); \
    if (dn_raw) std::copy((o)->link_dn.begin(), (o)->link_dn.end(), dn_raw); \
    if (up) std::copy((o)->link_up_c.begin(), (o)->link_up_c.end(), up); \
    if (dn) std::copy((o)->link_dn_c.begin(), (o)->link_dn_c.end(), dn); \
    if (start) std::copy((o)->start_hit.begin(), (o)->start_hit.end(), start); } while (0)
  if (h->precision == 0) GL(h->f); else GL(h->d);
#undef GL
}
// par: [n_tracks][5], cov: [n_tracks][15] (row-major per track), ints: [n_tracks][5] =
// n_hits, n_fit, first_row, last_row, start_hit
void oracle_get_tracks(void* hv, double* x_ref, double* z_ref, double* par, double* cov, double* chi2,
                       int32_t* ints, int32_t* hit_offset, int32_t* hit_idx) {
  Handle* h = (Handle*)hv;
#define GT(o) do { \
    for (size_t t = 0; t < (o)->tracks.size(); ++t) { \
      const auto& T = (o)->tracks[t]; \
      x_ref[t] = (double)T.x_ref; z_ref[t] = (double)T.z_ref; chi2[t] = (double)T.chi2; \
      for (int i = 0; i < 5; ++i) par[t * 5 + i] = (double)T.p[i]; \
      for (int i = 0; i < 15; ++i) cov[t * 15 + i] = (double)T.C[i]; \
      ints[t * 5 + 0] = T.n_hits; ints[t * 5 + 1] = T.n_fit; ints[t * 5 + 2] = T.first_row; \
      ints[t * 5 + 3] = T.last_row; ints[t * 5 + 4] = T.start_hit; } \
    std::copy((o)->hit_offset.begin(), (o)->hit_offset.end(), hit_offset); \
    std::copy((o)->hit_idx.begin(), (o)->hit_idx.end(), hit_idx); } while (0)
  if (h->precision == 0) GT(h->f); else GT(h->d);
#undef GT
}

// S6 outputs of the last run with stage bit 32: owner [n_clusters], n_own [n_tracks], selected [n_selected]
int64_t oracle_n_selected(void* hv) {
  Handle* h = (Handle*)hv;
  return h->precision == 0 ? (int64_t)h->f->selected.size() : (int64_t)h->d->selected.size();
}
void oracle_get_selection(void* hv, int32_t* owner, int32_t* n_own, int32_t* selected) {
  Handle* h = (Handle*)hv;
#define GS(o) do { \
    std::copy((o)->owner.begin(), (o)->owner.end(), owner); \
    std::copy((o)->n_own.begin(), (o)->n_own.end(), n_own); \
    std::copy((o)->selected.begin(), (o)->selected.end(), selected); } while (0)
  if (h->precision == 0) GS(h->f); else GS(h->d);
#undef GS
}
// S8: match and refit across the sectors held by `handles` (each after a run with stage bits up to 64)
int oracle_merge(void** handles, int n_sectors) {
  if (n_sectors <= 0) return 0;
  const int prec = ((Handle*)handles[0])->precision;
  if (prec == 0) {
    std::vector<Oracle<float>*> S;
    for (int i = 0; i < n_sectors; ++i) S.push_back(((Handle*)handles[i])->f);
    merge_sectors(S);
  } else {
    std::vector<Oracle<double>*> S;
    for (int i = 0; i < n_sectors; ++i) S.push_back(((Handle*)handles[i])->d);
    merge_sectors(S);
  }
  return 0;
}
// TEST HOOK for the S8 decision pins: replace the sector's selected tracks by hand-made ones (no clusters, no hit lists:
// the chain refit then has nothing to fit).  Per track: ints = first_row, last_row, out_ok; ref = x_ref, z_ref;
// par[5] = fitted state at x_ref; out[6] = outer state x, p0..p4.  No arithmetic happens here.
void oracle_inject_selected(void* hv, int32_t n, const int32_t* ints, const double* ref, const double* par, const double* out) {
  Handle* h = (Handle*)hv;
#define INJ(o, R) do { \
    (o)->n = 0; (o)->tracks.clear(); (o)->selected.clear(); (o)->out_state.clear(); (o)->out_ok.clear(); \
    (o)->hit_offset.assign(1, 0); (o)->hit_idx.clear(); \
    for (int32_t i = 0; i < n; ++i) { \
      Track<R> t{}; t.x_ref = (R)ref[2 * i]; t.z_ref = (R)ref[2 * i + 1]; \
      for (int q = 0; q < 5; ++q) t.p[q] = (R)par[5 * i + q]; \
      t.first_row = ints[3 * i]; t.last_row = ints[3 * i + 1]; t.n_hits = 0; t.n_fit = 0; t.start_hit = -1; \
      (o)->tracks.push_back(t); (o)->selected.push_back(i); (o)->hit_offset.push_back(0); \
      KFState<R> st{}; st.x = (R)out[6 * i]; for (int q = 0; q < 5; ++q) st.p[q] = (R)out[6 * i + 1 + q]; \
      for (int q = 0; q < 15; ++q) { st.C[q] = (R)0; } \
      st.chi2 = (R)0; st.n = 0; \
      (o)->out_state.push_back(st); (o)->out_ok.push_back((char)ints[3 * i + 2]); } } while (0)
  if (h->precision == 0) INJ(h->f, float); else INJ(h->d, double);
#undef INJ
}
// per selected track of the sector: partner above / below; returns the number of merged chains headed here and
// (out[1]) the total number of their segments
void oracle_get_merge_links(void* hv, int32_t* next_sec, int32_t* next_trk, int32_t* prev_sec, int32_t* prev_trk, int64_t* out) {
  Handle* h = (Handle*)hv;
#define GM(o) do { \
    std::copy((o)->mg_next_sec.begin(), (o)->mg_next_sec.end(), next_sec); std::copy((o)->mg_next_trk.begin(), (o)->mg_next_trk.end(), next_trk); \
    std::copy((o)->mg_prev_sec.begin(), (o)->mg_prev_sec.end(), prev_sec); std::copy((o)->mg_prev_trk.begin(), (o)->mg_prev_trk.end(), prev_trk); \
    out[0] = (int64_t)(o)->merged.size(); out[1] = 0; for (auto& m : (o)->merged) out[1] += (int64_t)m.seg_sec.size(); } while (0)
  if (h->precision == 0) GM(h->f); else GM(h->d);
#undef GM
}
// merged chains headed in this sector: ints [n][6] = head (selected index), n_seg, n_hits, n_fit, first_row, last_row + frame segment;
// seg_offset [n + 1], seg_sec / seg_trk [total segments]
void oracle_get_merged(void* hv, int32_t* ints, double* x_ref, double* z_ref, double* par, double* cov, double* chi2,
                       int32_t* seg_offset, int32_t* seg_sec, int32_t* seg_trk) {
  Handle* h = (Handle*)hv;
#define GG2(o) do { \
    int32_t off = 0; size_t i = 0; \
    for (auto& m : (o)->merged) { \
      ints[i * 7 + 0] = m.head; ints[i * 7 + 1] = (int32_t)m.seg_sec.size(); ints[i * 7 + 2] = m.t.n_hits; ints[i * 7 + 3] = m.t.n_fit; \
      ints[i * 7 + 4] = m.t.first_row; ints[i * 7 + 5] = m.t.last_row; ints[i * 7 + 6] = m.t.start_hit; \
      x_ref[i] = (double)m.t.x_ref; z_ref[i] = (double)m.t.z_ref; chi2[i] = (double)m.t.chi2; \
      for (int q = 0; q < 5; ++q) par[i * 5 + q] = (double)m.t.p[q]; \
      for (int q = 0; q < 15; ++q) cov[i * 15 + q] = (double)m.t.C[q]; \
      seg_offset[i] = off; \
      for (size_t q = 0; q < m.seg_sec.size(); ++q) { seg_sec[off] = m.seg_sec[q]; seg_trk[off] = m.seg_trk[q]; ++off; } \
      ++i; } \
    seg_offset[i] = off; } while (0)
  if (h->precision == 0) GG2(h->f); else GG2(h->d);
#undef GG2
}
// unit entry point for the pins: rotate a state [x, p0..p4, C0..C14, chi2] by (ca, sa)
int oracle_kf_rotate(void* hv, double* st, double ca, double sa) {
  Handle* h = (Handle*)hv;
  if (h->precision == 0) { KFState<float> s; st_in(s, st); bool ok = h->f->rotate(s, (float)ca, (float)sa); st_out(s, st); return ok; }
  KFState<double> s; st_in(s, st); bool ok = h->d->rotate(s, ca, sa); st_out(s, st); return ok;
}

// S7 outputs of the last run with stage bit 64, per cluster: res_trk i32, res_y / res_z double, q_y / q_z i16
void oracle_get_residuals(void* hv, int32_t* res_trk, double* res_y, double* res_z, int16_t* q_y, int16_t* q_z) {
  Handle* h = (Handle*)hv;
#define GR(o) do { \
    std::copy((o)->res_trk.begin(), (o)->res_trk.end(), res_trk); \
    copy_out(res_y, (o)->res_y); copy_out(res_z, (o)->res_z); \
    std::copy((o)->q_y.begin(), (o)->q_y.end(), q_y); std::copy((o)->q_z.begin(), (o)->q_z.end(), q_z); } while (0)
  if (h->precision == 0) GR(h->f); else GR(h->d);
#undef GR
}
// the selector on its own, on hit lists given by the caller (pins): returns the number of selected tracks
int64_t oracle_select(int64_t n_clusters, int64_t n_tracks, const int32_t* hit_offset, const int32_t* hit_idx,
                      int32_t max_shared_permille, int32_t* owner, int32_t* n_own, int32_t* selected) {
  std::vector<int32_t> o, w, s;
  select_tracks_plain(n_clusters, n_tracks, hit_offset, hit_idx, max_shared_permille, o, w, s);
  std::copy(o.begin(), o.end(), owner);
  std::copy(w.begin(), w.end(), n_own);
  std::copy(s.begin(), s.end(), selected);
  return (int64_t)s.size();
}

// ---- unit entry points for the pins ---------------------------------------------------
// state = [x, p0..p4, C0..C14, chi2] (22 doubles), in/out
int oracle_kf_propagate(void* hv, double* st, double x2) {
  Handle* h = (Handle*)hv;
  if (h->precision == 0) { KFState<float> s; st_in(s, st); bool ok = h->f->propagate(s, (float)x2); st_out(s, st); return ok; }
  KFState<double> s; st_in(s, st); bool ok = h->d->propagate(s, x2); st_out(s, st); return ok;
}
void oracle_kf_update(void* hv, double* st, double ym, double zm) {
  Handle* h = (Handle*)hv;
  if (h->precision == 0) { KFState<float> s; st_in(s, st); h->f->update(s, (float)ym, (float)zm); st_out(s, st); return; }
  KFState<double> s; st_in(s, st); h->d->update(s, ym, zm); st_out(s, st);
}
double oracle_kf_dist2(void* hv, const double* st, double ym, double zm) {
  Handle* h = (Handle*)hv;
  if (h->precision == 0) { KFState<float> s; st_in(s, st); return (double)h->f->dist2(s, (float)ym, (float)zm); }
  KFState<double> s; st_in(s, st); return h->d->dist2(s, ym, zm);
}
// S2 score of the triplet (d, c, u) around row r with the oracle's arithmetic (reading N4)
double oracle_score(void* hv, int r, double yc, double zc, double yu, double zu, double yd, double zd) {
  Handle* h = (Handle*)hv;
  if (h->precision == 0)
    return (double)h->f->score(r, (float)yc, (float)zc, (float)yu, (float)zu, (float)yd, (float)zd);
  return h->d->score(r, yc, zc, yu, zu, yd, zd);
}

}  // extern "C"
