"""Pins of the CPU oracle.

The paper prints no value for this path, so the oracle is pinned to what the
mathematics fixes: invariants, brute force on tiny inputs, closed forms (second difference
of a parabola, weighted least squares), exact special cases (straight lines on a dyadic
geometry, exact helices from circle geometry), statistics (unit pulls) and generator truth.
None of these re-use the oracle's own formulae.
"""
import math

import numpy as np
import pytest

import tpcsynth
from tpcsynth.truth import sector_metrics, summarize
from oracle import Oracle, run_timeframe


# ----------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------
def links_in_original_ids(res):
    """(up, dn) links indexed and valued by ORIGINAL cluster id (-1 = none)."""
    n = res.n
    up = np.full(n, -1, np.int64)
    dn = np.full(n, -1, np.int64)
    o = res.order.astype(np.int64)
    m = res.link_up_raw >= 0
    up[o[m]] = o[res.link_up_raw[m]]
    m = res.link_dn_raw >= 0
    dn[o[m]] = o[res.link_dn_raw[m]]
    return up, dn


def dense_random_sector(params, n, seed, zmax=40.0, rows=None):
    """Uniform random clusters, dense enough that windows hold several candidates."""
    rng = np.random.default_rng(seed)
    nr = params.n_rows if rows is None else rows
    row = rng.integers(0, nr, n).astype(np.uint16)
    y = (rng.random(n) * 16.0 - 8.0).astype(np.float32)
    z = (rng.random(n) * zmax).astype(np.float32)
    return y, z, row


# ----------------------------------------------------------------------------------------
# P1  S1 grid invariants
# ----------------------------------------------------------------------------------------
def test_p1_grid_invariants(cfg0):
    tf = cfg0
    P = tf.params
    res = run_timeframe(tf, stage_mask=1)[0]
    n = res.n
    assert sorted(res.order.tolist()) == list(range(n))                 # a permutation
    assert np.all(np.diff(res.bin_start.astype(np.int64)) >= 0)         # monotone
    assert res.bin_start[0] == 0 and res.bin_start[-1] == n
    assert res.bin_start.shape[0] == P.bins_per_sector() + 1
    # recompute every cluster's bin independently (numpy fp32, same data tables)
    y = tf.y[0][res.order]; z = tf.z[0][res.order]; r = tf.row[0][res.order].astype(np.int64)
    assert np.array_equal(res.sy.astype(np.float32), y) and np.array_equal(res.sz.astype(np.float32), z)
    by = np.clip(np.floor((y - P.grid_y_lo[r]) * P.grid_inv_bin_y[r]), 0, P.grid_ny[r] - 1).astype(np.int64)
    bz = np.clip(np.floor((z - np.float32(P.grid_z_lo)) * P.grid_inv_bin_z[r]), 0, P.grid_nz[r] - 1).astype(np.int64)
    base = np.concatenate([[0], np.cumsum(P.grid_ny.astype(np.int64) * P.grid_nz)])
    g = base[r] + bz * P.grid_ny[r] + by
    assert np.all(np.diff(g) >= 0)                                      # sorted by (row, bin)
    pos = np.arange(n)
    assert np.all(res.bin_start[g] <= pos) and np.all(pos < res.bin_start[g + 1])
    same = np.diff(g) == 0
    assert np.all(np.diff(res.order)[same] > 0)                         # ids ascending inside a bin
    assert np.array_equal(res.row_start, np.searchsorted(r, np.arange(P.n_rows + 1)).astype(np.int32))


def test_p1_clusters_outside_grid_are_clamped(cfg0):
    """Reading N9: clusters outside the grid range land in edge bins, never dropped."""
    P = cfg0.params
    y = np.array([-1e3, 1e3, 0.0, 0.0], np.float32)
    z = np.array([10.0, 10.0, -50.0, 1e6], np.float32)
    row = np.array([5, 5, 5, 5], np.uint16)
    res = Oracle(P).run(y, z, row, stage_mask=1)
    assert res.bin_start[-1] == 4 and sorted(res.order.tolist()) == [0, 1, 2, 3]


# ----------------------------------------------------------------------------------------
# P2  S2: grid search == brute force all pairs (oracle brute mode AND independent numpy)
# ----------------------------------------------------------------------------------------
def numpy_all_pairs_links(P, y, z, row):
    """All-pairs neighbour search in numpy fp32, original-id space; independent of the grid."""
    f = np.float32
    n = y.shape[0]
    up = np.full(n, -1, np.int64); dn = np.full(n, -1, np.int64)
    ids_by_row = [np.nonzero(row == r)[0] for r in range(P.n_rows)]
    for c in range(n):
        r = int(row[c])
        if r < 1 or r > P.n_rows - 2:
            continue
        U = ids_by_row[r + 1]; D = ids_by_row[r - 1]
        U = U[(np.abs(y[U] - y[c]) <= P.nf_hy_up[r]) & (np.abs(z[U] - z[c]) <= P.nf_hz_up[r])]
        D = D[(np.abs(y[D] - y[c]) <= P.nf_hy_dn[r]) & (np.abs(z[D] - z[c]) <= P.nf_hz_dn[r])]
        if U.size == 0 or D.size == 0:
            continue
        dxu = f(P.row_x[r + 1] - P.row_x[r]); dxd = f(P.row_x[r] - P.row_x[r - 1])
        ay = ((y[U] - y[c]) * dxd)[:, None] - ((y[c] - y[D]) * dxu)[None, :]
        az = ((z[U] - z[c]) * dxd)[:, None] - ((z[c] - z[D]) * dxu)[None, :]
        s = ay * ay + az * az
        assert s.dtype == np.float32
        m = s.min()
        cand = np.argwhere(s == m)
        # ties: smallest original id of u, then of d (U, D are ascending in id)
        iu, idn = min((int(U[a]), int(D[b])) for a, b in cand)
        if m <= P.nf_cut[r]:
            up[c] = iu; dn[c] = idn
    return up, dn


@pytest.mark.parametrize("seed", [1, 2])
def test_p2_brute_force_neighbours(seed):
    P = tpcsynth.default_params(n_sectors=1)
    y, z, row = dense_random_sector(P, 2000, seed, zmax=30.0, rows=12)
    orc = Oracle(P)
    grid = orc.run(y, z, row, stage_mask=3)
    brute = orc.run(y, z, row, stage_mask=3, brute=True)
    assert np.array_equal(grid.link_up_raw, brute.link_up_raw)
    assert np.array_equal(grid.link_dn_raw, brute.link_dn_raw)
    up, dn = links_in_original_ids(grid)
    up_np, dn_np = numpy_all_pairs_links(P, y, z, row)
    assert (up >= 0).sum() > 200                       # the case is not vacuous
    assert np.array_equal(up, up_np) and np.array_equal(dn, dn_np)


def test_p2_brute_force_on_config0(cfg0):
    tf = cfg0
    orc = Oracle(tf.params)
    a = orc.run(tf.y[0], tf.z[0], tf.row[0], stage_mask=3)
    b = orc.run(tf.y[0], tf.z[0], tf.row[0], stage_mask=3, brute=True)
    assert np.array_equal(a.link_up_raw, b.link_up_raw) and np.array_equal(a.link_dn_raw, b.link_dn_raw)
    assert (a.link_up_raw >= 0).sum() > 3000


def test_p2_ties_and_duplicates():
    """Reading N7: duplicated clusters are legal; ties go to the smallest original id."""
    P = tpcsynth.default_params(n_sectors=1)
    # rows 9,10,11: two identical up candidates (ids 3, 1) and two identical down candidates (ids 4, 2)
    y = np.array([0.0, 0.5, -0.5, 0.5, -0.5], np.float32)
    z = np.array([10.0, 10.5, 9.5, 10.5, 9.5], np.float32)
    row = np.array([10, 11, 9, 11, 9], np.uint16)
    res = Oracle(P).run(y, z, row, stage_mask=3)
    up, dn = links_in_original_ids(res)
    assert up[0] == 1 and dn[0] == 2


# ----------------------------------------------------------------------------------------
# closed form for the S2 score: second difference of a parabola
# ----------------------------------------------------------------------------------------
def test_score_closed_form_parabola():
    """For y = a + b x + c x^2 the collinearity residual is exactly c*dxu*dxd*(dxu+dxd)
    (divided differences); with dyadic numbers fp32 reproduces it exactly.  Pins signs,
    operand order and the use of dxu/dxd in the score."""
    row_x = 64.0 + np.array([0.0, 0.5, 1.5, 1.75])          # unequal pitches
    P = tpcsynth.default_params(n_sectors=1, row_x=row_x)
    orc = Oracle(P)
    a, b, c = 1.0, 0.25, 0.125
    ea, eb, ec = -2.0, 0.5, -0.0625
    yf = lambda x: a + b * x + c * x * x
    zf = lambda x: ea + eb * x + ec * x * x
    for r in (1, 2):
        xd, xc, xu = row_x[r - 1] - 64.0, row_x[r] - 64.0, row_x[r + 1] - 64.0
        dxu, dxd = xu - xc, xc - xd
        ay = c * dxu * dxd * (dxu + dxd)
        az = ec * dxu * dxd * (dxu + dxd)
        s = orc.score(r, yf(xc), zf(xc), yf(xu), zf(xu), yf(xd), zf(xd))
        assert s == ay * ay + az * az
    # collinear -> exactly zero; swapping u and d must NOT be symmetric when dxu != dxd
    s0 = orc.score(1, 1.0, 2.0, 1.0 + 0.25 * 1.0, 2.0 + 1.0, 1.0 - 0.25 * 0.5, 2.0 - 0.5)
    assert s0 == 0.0
    s1 = orc.score(1, 1.0, 2.0, 1.0 - 0.25 * 0.5, 2.0 - 0.5, 1.0 + 0.25 * 1.0, 2.0 + 1.0)
    assert s1 > 0.0


# ----------------------------------------------------------------------------------------
# P3  metamorphic: links do not depend on the grid; y-mirror symmetry
# ----------------------------------------------------------------------------------------
def test_p3_links_independent_of_grid_and_mirror():
    tf = tpcsynth.generate(1, n_tracks=600)
    s = 3
    y, z, row = tf.y[s], tf.z[s], tf.row[s]
    base = Oracle(tf.params).run(y, z, row, stage_mask=3)
    up0, dn0 = links_in_original_ids(base)
    assert (up0 >= 0).sum() > 1000
    for bs, gm in ((0.5, 0.01), (1.7, 0.01), (3.0, 0.5), (1.0, 0.0625)):
        P2 = tpcsynth.default_params(n_sectors=36, bin_scale=bs, grid_margin=gm)
        r2 = Oracle(P2).run(y, z, row, stage_mask=3)
        up, dn = links_in_original_ids(r2)
        assert np.array_equal(up, up0) and np.array_equal(dn, dn0), (bs, gm)
    rm = Oracle(tf.params).run(-y, z, row, stage_mask=3)        # negation is exact
    up, dn = links_in_original_ids(rm)
    assert np.array_equal(up, up0) and np.array_equal(dn, dn0)


# ----------------------------------------------------------------------------------------
# hand-worked toy (tests/golden/toy_links.txt): S2 cut, S3 reciprocity, S4 start hits
# ----------------------------------------------------------------------------------------
def test_toy_worked_example():
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "toy_links.txt")
    rows, ys, zs, exp_up, exp_dn, exp_upc, exp_dnc = [], [], [], [], [], [], []
    exp_start = None
    for line in open(path):
        line = line.split("#")[0].strip()
        if not line:
            continue
        if line.startswith("start"):
            exp_start = [int(v) for v in line.split()[1:]]
            continue
        f = line.split()
        rows.append(int(f[1])); ys.append(float(f[2])); zs.append(float(f[3]))
        exp_up.append(int(f[4])); exp_dn.append(int(f[5])); exp_upc.append(int(f[6])); exp_dnc.append(int(f[7]))
    row_x = 64.0 + 1.0 * np.arange(8)
    P = tpcsynth.default_params(n_sectors=1, row_x=row_x, sigma=0.125)
    res = Oracle(P).run(np.array(ys, np.float32), np.array(zs, np.float32), np.array(rows, np.uint16), stage_mask=0xF)
    o = res.order.astype(np.int64)

    def to_orig(a):
        out = np.full(res.n, -1, np.int64)
        m = a >= 0
        out[o[m]] = o[a[m]]
        return out
    assert to_orig(res.link_up_raw).tolist() == exp_up
    assert to_orig(res.link_dn_raw).tolist() == exp_dn
    assert to_orig(res.link_up).tolist() == exp_upc
    assert to_orig(res.link_dn).tolist() == exp_dnc
    assert sorted(o[res.start_hit].tolist()) == sorted(exp_start)


# ----------------------------------------------------------------------------------------
# P4  exact recovery of noise-free straight tracks on a dyadic geometry
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", ["f32", "f64"])
def test_p4_straight_tracks_exact(precision):
    row_x = 64.0 + 0.75 * np.arange(152)
    P = tpcsynth.default_params(n_sectors=1, row_x=row_x)
    nt = 12
    y0 = -6.0 + 1.0 * np.arange(nt)                  # 1 cm apart at row 0
    ty = (np.arange(nt) - 6) / 64.0                  # dyadic slopes, fan out
    z0 = 8.0 + 16.0 * np.arange(nt)                  # well separated in z
    tz = (np.arange(nt) - 4) / 8.0
    row, y, z, trk = tpcsynth.straight_tracks(row_x, y0, ty, z0, tz)
    rng = np.random.default_rng(5)
    perm = rng.permutation(row.shape[0])
    row, y, z, trk = row[perm], y[perm], z[perm], trk[perm]
    assert np.array_equal(y.astype(np.float32).astype(np.float64), y)   # exactly representable
    orc = Oracle(P, precision)
    res = orc.run(y, z, row)
    lab = trk[res.order]
    srow = row[res.order]
    # every S2 score is exactly zero -> every interior cluster is linked to its own track
    inner = (srow >= 1) & (srow <= 150)
    assert np.all(res.link_up_raw[inner] >= 0) and np.all(res.link_dn_raw[inner] >= 0)
    assert np.array_equal(lab[res.link_up_raw[inner]], lab[inner])
    assert np.array_equal(lab[res.link_dn_raw[inner]], lab[inner])
    assert np.array_equal(srow[res.link_up_raw[inner]], srow[inner] + 1)
    for c in np.nonzero(inner)[0][::97]:
        u, d = res.link_up_raw[c], res.link_dn_raw[c]
        assert orc.score(int(srow[c]), res.sy[c], res.sz[c], res.sy[u], res.sz[u], res.sy[d], res.sz[d]) == 0.0
    # rows 0 and 151 own no links (reading N2); chains run 1..150; one start hit per track at row 1
    assert np.all(res.link_up_raw[~inner] == -1) and np.all(res.link_dn_raw[~inner] == -1)
    assert len(res.start_hit) == nt and np.all(srow[res.start_hit] == 1)
    assert res.n_tracks == nt
    for t in range(nt):
        hits = res.hit_idx[res.hit_offset[t]:res.hit_offset[t + 1]]
        assert len(hits) == 152 and res.first_row[t] == 0 and res.last_row[t] == 151
        k = lab[hits[0]]
        assert np.all(lab[hits] == k) and np.array_equal(srow[hits], np.arange(152))
        tol = 2e-5 if precision == "f32" else 1e-9
        norm = math.sqrt(1.0 + ty[k] ** 2)
        assert res.x_ref[t] == row_x[0]
        assert abs(res.par[t, 0] - y0[k]) < tol * 10
        assert abs(res.z_ref[t] + res.par[t, 1] - z0[k]) < tol * 100
        assert abs(res.par[t, 2] - ty[k] / norm) < tol
        assert abs(res.par[t, 3] - tz[k] / norm) < tol * 10
        assert abs(res.par[t, 4]) < (2e-3 if precision == "f32" else 1e-7)   # 1/pT = 0
        assert res.chi2[t] < (1e-4 if precision == "f32" else 1e-12)


# ----------------------------------------------------------------------------------------
# P5  S3/S4 invariants
# ----------------------------------------------------------------------------------------
def test_p5_link_invariants(cfg1_small):
    tf = cfg1_small
    for s in (0, 7, 25):
        res = run_timeframe(tf, sectors=[s], stage_mask=0xF)[s]
        n = res.n
        c = np.arange(n)
        up, dn = res.link_up, res.link_dn
        m = up >= 0
        assert np.array_equal(dn[up[m]], c[m])                    # reciprocal both ways
        m2 = dn >= 0
        assert np.array_equal(up[dn[m2]], c[m2])
        assert m.sum() == m2.sum()
        srow = tf.row[s][res.order].astype(np.int64)
        assert np.all(srow[up[m]] == srow[m] + 1)                 # consecutive rows
        # cleaned links are a subset of the raw ones
        assert np.all(res.link_up_raw[m] == up[m]) and np.all(res.link_dn_raw[m2] == dn[m2])
        start = (dn == -1) & (up >= 0)
        end = (up == -1) & (dn >= 0)
        assert np.array_equal(np.nonzero(start)[0], res.start_hit)    # ascending sorted index
        assert start.sum() == end.sum()                           # #start hits == #chain ends
        # every chain is a simple path: following up from the start hits visits each linked cluster once
        seen = np.zeros(n, bool)
        cur = res.start_hit.copy()
        while cur.size:
            assert not seen[cur].any()
            seen[cur] = True
            cur = up[cur]
            cur = cur[cur >= 0]
        assert np.array_equal(seen, (up >= 0) | (dn >= 0))


# ----------------------------------------------------------------------------------------
# transport: exact circle geometry, finite-difference Jacobian
# ----------------------------------------------------------------------------------------
def _state(x, p, C=None, chi2=0.0):
    st = np.zeros(22)
    st[0] = x; st[1:6] = p
    if C is not None:
        st[6:21] = C
    st[21] = chi2
    return st


def test_propagate_follows_exact_helix():
    """Parameter transport vs the exact circle (generator geometry: asin/sqrt in double)."""
    P = tpcsynth.default_params(n_sectors=1)
    orc = Oracle(P, "f64")
    row_x = P.row_x.astype(np.float64)
    Bc = float(P.kappa_per_qpt)
    for sp0, p4, dzds in ((0.1, 1.0, 0.4), (-0.3, -2.5, -0.9), (0.6, -4.0, 0.2), (0.0, 0.15, 1.0)):
        kappa = p4 * Bc
        rows, y, z, sp = tpcsynth.helix_hits(row_x, row_x[0], 3.0, 0.0, sp0, dzds, kappa)
        st = _state(row_x[0], [3.0, 0.0, sp0, dzds, p4])
        for r in rows[1:]:                       # row by row
            if abs(sp[list(rows).index(r)]) > 0.94:
                break
            ok, st = orc.kf_propagate(st, row_x[r])
            assert ok
            i = list(rows).index(r)
            assert abs(st[1] - y[i]) < 1e-9 * max(1.0, abs(y[i]))
            assert abs(st[2] - z[i]) < 1e-9 * max(1.0, abs(z[i]))
            assert abs(st[3] - sp[i]) < 1e-12
        # one long step up and back down returns to the start
        far = rows[min(len(rows) - 1, 60)]
        if abs(sp[list(rows).index(far)]) < 0.94:
            ok, s2 = orc.kf_propagate(_state(row_x[0], [3.0, 0.0, sp0, dzds, p4]), row_x[far])
            i = list(rows).index(far)
            # arc = chord*(1 + t/24 + 3t^2/640), t = (k d)^2: truncation <= 2*(5/7168)*(k d)^6 relative
            d = math.hypot(row_x[far] - row_x[0], y[i] - 3.0)
            tol_z = 1e-9 + abs(dzds) * d * 2.0 * (5.0 / 7168.0) * (kappa * d) ** 6
            assert ok and abs(s2[1] - y[i]) < 1e-9 and abs(s2[2] - z[i]) < tol_z
            ok, s3 = orc.kf_propagate(s2, row_x[0])
            assert ok and abs(s3[1] - 3.0) < 1e-9 and abs(s3[2]) < 1e-9 and abs(s3[3] - sp0) < 1e-12


def test_propagate_fails_beyond_max_sinphi_and_leaves_state():
    P = tpcsynth.default_params(n_sectors=1)
    orc = Oracle(P, "f32")
    st = _state(100.0, [0.0, 0.0, 0.9, 0.1, 6.0], C=np.arange(15) * 0.01)
    ok, s2 = orc.kf_propagate(st, 130.0)            # sin(phi) would reach 0.9 + 6*Bc*30 = 1.17
    assert not ok and np.array_equal(s2, st.astype(np.float32).astype(np.float64))
    ok, s3 = orc.kf_propagate(st, 100.0)            # dx = 0: no-op success
    assert ok and np.array_equal(s3, st.astype(np.float32).astype(np.float64))


def test_jacobian_finite_differences():
    """C' = J C J^T with C = e_j e_j^T gives column j of J; compare with central differences
    of the parameter transport itself.  n02, n04, n13, n24 are exact derivatives; n12 and n14
    are leading-order, checked to 2 %."""
    P = tpcsynth.default_params(n_sectors=1)
    orc = Oracle(P, "f64")
    x1, x2 = 100.0, 104.5
    p = np.array([2.0, -1.0, 0.25, 0.7, -1.2])

    def transport(q):
        ok, s = orc.kf_propagate(_state(x1, q), x2)
        assert ok
        return s[1:6]
    J_fd = np.zeros((5, 5))
    for j in range(5):
        h = 1e-6
        dp = np.zeros(5); dp[j] = h
        J_fd[:, j] = (transport(p + dp) - transport(p - dp)) / (2 * h)
    J_cov = np.zeros((5, 5))
    tri = lambda i, j: i * (i + 1) // 2 + j
    for j in range(5):
        C = np.zeros(15); C[tri(j, j)] = 1.0
        ok, s = orc.kf_propagate(_state(x1, p, C), x2)
        Cn = s[6:21]
        col = np.array([Cn[tri(max(i, j), min(i, j))] for i in range(5)])   # = J[i,j]*J[j,j], J[j,j] = 1
        J_cov[:, j] = col
    exact = [(0, 0), (1, 1), (2, 2), (3, 3), (4, 4), (0, 2), (0, 4), (1, 3), (2, 4)]
    for (i, j) in exact:
        assert abs(J_cov[i, j] - J_fd[i, j]) < 1e-6 * max(1.0, abs(J_fd[i, j])), (i, j)
    for (i, j) in [(1, 2), (1, 4)]:
        assert abs(J_cov[i, j] - J_fd[i, j]) < 0.02 * abs(J_fd[i, j]) + 1e-9, (i, j)
    zero = [(i, j) for i in range(5) for j in range(5) if (i, j) not in exact + [(1, 2), (1, 4)]]
    for (i, j) in zero:
        assert J_cov[i, j] == 0.0 and abs(J_fd[i, j]) < 1e-6, (i, j)


def test_update_is_the_textbook_scalar_kalman_update():
    """One measurement update vs the matrix form K = C H^T (H C H^T + V)^-1 computed in numpy
    (sequential scalar updates of uncorrelated measurements equal the joint update)."""
    P = tpcsynth.default_params(n_sectors=1)
    orc = Oracle(P, "f64")
    rng = np.random.default_rng(3)
    A = rng.standard_normal((5, 5))
    Cm = A @ A.T + np.eye(5)
    tri = [(i, j) for i in range(5) for j in range(i + 1)]
    C = np.array([Cm[i, j] for i, j in tri])
    p = rng.standard_normal(5)
    ym, zm = 0.3, -0.7
    st = orc.kf_update(_state(90.0, p, C), ym, zm)
    H = np.zeros((2, 5)); H[0, 0] = 1; H[1, 1] = 1
    V = np.diag([P.err2_y, P.err2_z])
    S = H @ Cm @ H.T + V
    K = Cm @ H.T @ np.linalg.inv(S)
    r = np.array([ym, zm]) - H @ p
    p_ref = p + K @ r
    C_ref = Cm - K @ H @ Cm
    chi2_ref = r @ np.linalg.inv(S) @ r
    assert np.allclose(st[1:6], p_ref, rtol=1e-10, atol=1e-12)
    assert np.allclose(st[6:21], [C_ref[i, j] for i, j in tri], rtol=1e-9, atol=1e-12)
    assert abs(st[21] - chi2_ref) < 1e-10
    d2 = orc.kf_dist2(_state(90.0, p, C), ym, zm)
    assert abs(d2 - (r[0] ** 2 / S[0, 0] + r[1] ** 2 / S[1, 1])) < 1e-12


# ----------------------------------------------------------------------------------------
# P6  noise-free helices: fitted parameters equal truth (1e-5 relative in double)
# ----------------------------------------------------------------------------------------
def _helix_sector(P, tracks, dtype):
    row_x = P.row_x.astype(np.float64)
    ys, zs, rows, labs, truth = [], [], [], [], []
    for t, (y0, z0, sp0, dzds, p4) in enumerate(tracks):
        rr, y, z, sp = tpcsynth.helix_hits(row_x, row_x[0], y0, z0, sp0, dzds, p4 * float(P.kappa_per_qpt))
        keep = np.abs(sp) < 0.9
        rr, y, z = rr[keep], y[keep], z[keep]
        ys.append(y); zs.append(z); rows.append(rr); labs.append(np.full(len(rr), t))
    y = np.concatenate(ys); z = np.concatenate(zs); row = np.concatenate(rows).astype(np.uint16)
    lab = np.concatenate(labs)
    perm = np.random.default_rng(11).permutation(len(y))
    return y[perm].astype(dtype), z[perm].astype(dtype), row[perm], lab[perm]


HELIX_TRACKS = [  # y0, z0, sin(phi0), dz/ds, q/pT
    (-9.0, 20.0, 0.05, 0.3, 0.2), (-4.0, 60.0, -0.10, -0.5, -0.8), (0.0, 100.0, 0.20, 0.9, 1.7),
    (4.0, 140.0, -0.30, 0.1, -3.0), (8.0, 180.0, 0.10, -1.0, 5.0), (11.0, 220.0, 0.0, 0.6, -0.15),
]


def test_p6_helix_recovery_double():
    P = tpcsynth.default_params(n_sectors=1)
    y, z, row, lab = _helix_sector(P, HELIX_TRACKS, np.float64)
    res = Oracle(P, "f64").run(y, z, row)
    assert res.n_tracks == len(HELIX_TRACKS)
    floors = np.array([1.0, 1.0, 0.1, 0.1, 0.1])
    for t in range(res.n_tracks):
        hits = res.hit_idx[res.hit_offset[t]:res.hit_offset[t + 1]]
        k = int(lab[res.order][hits[0]])
        y0, z0, sp0, dzds, p4 = HELIX_TRACKS[k]
        assert res.n_hits[t] == (lab == k).sum() and res.first_row[t] == 0
        got = np.array([res.par[t, 0], res.z_ref[t] + res.par[t, 1], res.par[t, 2], res.par[t, 3], res.par[t, 4]])
        want = np.array([y0, z0, sp0, dzds, p4])
        rel = np.abs(got - want) / np.maximum(np.maximum(np.abs(got), np.abs(want)), floors)
        assert np.all(rel < 1e-5), (k, rel)


def test_p6_helix_recovery_float():
    P = tpcsynth.default_params(n_sectors=1)
    y, z, row, lab = _helix_sector(P, HELIX_TRACKS, np.float32)
    res = Oracle(P, "f32").run(y, z, row)
    assert res.n_tracks == len(HELIX_TRACKS)
    floors = np.array([1.0, 1.0, 0.1, 0.1, 0.1])
    for t in range(res.n_tracks):
        hits = res.hit_idx[res.hit_offset[t]:res.hit_offset[t + 1]]
        k = int(lab[res.order][hits[0]])
        want = np.array(HELIX_TRACKS[k])
        got = np.array([res.par[t, 0], res.z_ref[t] + res.par[t, 1], res.par[t, 2], res.par[t, 3], res.par[t, 4]])
        rel = np.abs(got - want) / np.maximum(np.maximum(np.abs(got), np.abs(want)), floors)
        assert np.all(rel < 2e-3), (k, rel)      # fp32 cluster positions limit curvature


# ----------------------------------------------------------------------------------------
# P7  textbook reduction: weighted linear / quadratic least squares
# ----------------------------------------------------------------------------------------
def test_p7_wls_straight_line():
    """p4 frozen at 0 (init_cov[4] = 0).  (a) y exactly constant => phi == 0 exactly, path
    length == dx, and the z filter is *exactly* recursive linear regression of z on x;
    (b) z exactly constant (dz/ds == 0), small sigma => the y filter is linear regression of
    y on x with slope tan(phi).  Estimates, covariance and chi2 vs sigma^2 (X^T X)^-1."""
    tri = lambda i, j: i * (i + 1) // 2 + j
    # ---- (a) z fit
    sigma = 0.1
    P = tpcsynth.default_params(n_sectors=1, sigma=sigma)
    P.init_cov = np.array([1e4, 1e6, 1e2, 1e6, 0.0], np.float32)
    row_x = P.row_x.astype(np.float64)
    rng = np.random.default_rng(21)
    n = P.n_rows
    X = np.stack([np.ones(n), row_x - row_x[0]], axis=1)
    e2 = float(P.err2_z)                                   # the fp32-rounded sigma^2 the filter uses
    cov = e2 * np.linalg.inv(X.T @ X)
    y = np.full(n, 1.0)
    z = 50.0 + 0.8 * (row_x - row_x[0]) + sigma * rng.standard_normal(n)
    res = Oracle(P, "f64").run(y, z, np.arange(n, dtype=np.uint16))
    assert res.n_tracks == 1
    t = 0
    assert res.n_hits[t] == n and res.n_fit[t] == n and res.par[t, 2] == 0.0 and res.par[t, 0] == 1.0
    bz = np.linalg.lstsq(X, z, rcond=None)[0]
    assert abs(res.z_ref[t] + res.par[t, 1] - bz[0]) < 1e-5 * math.sqrt(cov[0, 0])
    assert abs(res.par[t, 3] - bz[1]) < 1e-5 * math.sqrt(cov[1, 1])
    C = res.cov[t]
    assert abs(C[tri(1, 1)] / cov[0, 0] - 1) < 1e-6
    assert abs(C[tri(3, 3)] / cov[1, 1] - 1) < 1e-6
    assert abs(C[tri(3, 1)] / cov[1, 0] - 1) < 1e-6
    rss = np.sum((z - X @ bz) ** 2)
    assert abs(res.chi2[t] / (rss / e2) - 1) < 1e-6
    # ---- (b) y fit
    sigma = 0.01
    P = tpcsynth.default_params(n_sectors=1, sigma=sigma)
    P.init_cov = np.array([1e4, 1e4, 1e2, 1e4, 0.0], np.float32)
    e2 = float(P.err2_y)
    cov = e2 * np.linalg.inv(X.T @ X)
    y = 1.0 + 0.05 * (row_x - row_x[0]) + sigma * rng.standard_normal(n)
    z = np.full(n, 50.0)
    res = Oracle(P, "f64").run(y, z, np.arange(n, dtype=np.uint16))
    assert res.n_tracks == 1 and res.n_hits[0] == n and res.par[0, 3] == 0.0
    by = np.linalg.lstsq(X, y, rcond=None)[0]
    cphi = 1.0 / math.sqrt(1.0 + by[1] ** 2)
    assert abs(res.par[0, 0] - by[0]) < 1e-3 * math.sqrt(cov[0, 0])
    assert abs(res.par[0, 2] - by[1] * cphi) < 1e-3 * math.sqrt(cov[1, 1]) * cphi ** 3
    C = res.cov[0]
    assert abs(C[tri(0, 0)] / cov[0, 0] - 1) < 1e-3
    assert abs(C[tri(2, 2)] / (cov[1, 1] * cphi ** 6) - 1) < 1e-3        # d sin/d tan = cos^3
    assert abs(C[tri(2, 0)] / (cov[1, 0] * cphi ** 3) - 1) < 1e-3


def test_p7_wls_parabola_curvature():
    """Small curvature with phi crossing zero, dz/ds == 0, small sigma: y(x) is a parabola up
    to O(phi^2) ~ 6e-5, so the fitted q/pT must equal the quadratic-regression curvature / Bc
    to a small fraction of its statistical error, with the same variance."""
    sigma = 0.01
    P = tpcsynth.default_params(n_sectors=1, sigma=sigma)
    P.init_cov = np.array([1e4, 1e4, 1e2, 1e4, 1e4], np.float32)
    row_x = P.row_x.astype(np.float64)
    Bc = float(P.kappa_per_qpt)
    kappa = 1e-4
    xm = 0.5 * (row_x[0] + row_x[-1])
    sp0 = -kappa * (xm - row_x[0])
    rows, y, z, sp = tpcsynth.helix_hits(row_x, row_x[0], 0.0, 30.0, sp0, 0.0, kappa)
    rng = np.random.default_rng(22)
    n = len(rows)
    assert n == P.n_rows and np.all(z == 30.0)
    y = y + sigma * rng.standard_normal(n)
    res = Oracle(P, "f64").run(y, z, rows.astype(np.uint16))
    assert res.n_tracks == 1 and res.n_hits[0] == n
    dx = row_x - row_x[0]
    X = np.stack([np.ones(n), dx, 0.5 * dx * dx], axis=1)
    b = np.linalg.lstsq(X, y, rcond=None)[0]
    cov = float(P.err2_y) * np.linalg.inv(X.T @ X)
    sig_k = math.sqrt(cov[2, 2])
    assert abs(res.par[0, 4] * Bc - b[2]) < 0.05 * sig_k
    assert abs(res.par[0, 2] - b[1]) < 0.05 * math.sqrt(cov[1, 1])
    assert abs(res.par[0, 0] - b[0]) < 0.05 * math.sqrt(cov[0, 0])
    tri = lambda i, j: i * (i + 1) // 2 + j
    assert abs(res.cov[0][tri(4, 4)] * Bc * Bc / cov[2, 2] - 1) < 0.01
    assert abs(res.cov[0][tri(4, 2)] * Bc / cov[2, 1] - 1) < 0.01
    assert abs(res.cov[0][tri(4, 0)] * Bc / cov[2, 0] - 1) < 0.01
    assert abs(res.par[0, 4] - kappa / Bc) < 4 * sig_k / Bc          # and it finds the truth


# ----------------------------------------------------------------------------------------
# P8 / P9 / P10  statistics and generator truth on config-1 kinematics
# ----------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def cfg1_tracks():
    tf = tpcsynth.generate(1, n_tracks=6000)
    secs = [0, 5, 11, 18, 23, 30]
    return tf, secs, run_timeframe(tf, sectors=secs)


def test_p8_pulls_and_chi2(cfg1_tracks):
    tf, secs, out = cfg1_tracks
    pulls, red = [], []
    tri = lambda i: i * (i + 1) // 2 + i
    for s in secs:
        res = out[s]
        lab = tf.label[s][res.order]
        for t in range(res.n_tracks):
            hits = res.hit_idx[res.hit_offset[t]:res.hit_offset[t + 1]]
            l = lab[hits]
            if res.n_hits[t] < 60 or l[0] < 0 or not np.all(l == l[0]) or res.n_fit[t] != res.n_hits[t]:
                continue
            tr = tpcsynth.truth_state(tf, int(l[0]), s, float(res.x_ref[t]))
            if tr is None:
                continue
            got = np.array([res.par[t, 0], res.z_ref[t] + res.par[t, 1], res.par[t, 2], res.par[t, 3], res.par[t, 4]])
            want = np.array([tr["y"], tr["z"], tr["sinphi"], tr["dzds"], tr["p4"]])
            err = np.sqrt(np.array([res.cov[t][tri(i)] for i in range(5)]))
            pulls.append((got - want) / err)
            red.append(res.chi2[t] / (2 * res.n_fit[t] - 5))
    pulls = np.array(pulls)
    assert pulls.shape[0] > 1500
    # clip the rare non-Gaussian tail (a wrong hit picked up) before taking moments
    core = np.all(np.abs(pulls) < 5, axis=1)
    assert core.mean() > 0.97
    pc = pulls[core]
    assert np.all(np.abs(pc.mean(axis=0)) < 0.1), pc.mean(axis=0)
    assert np.all(np.abs(pc.std(axis=0) - 1.0) < 0.1), pc.std(axis=0)
    assert abs(np.mean(np.array(red)[core]) - 1.0) < 0.05


def test_p9_covariance_sanity(cfg1_tracks):
    tf, secs, out = cfg1_tracks
    tri = lambda i, j: i * (i + 1) // 2 + j
    for s in secs:
        C = out[s].cov
        for i in range(5):
            assert np.all(C[:, tri(i, i)] > 0)
            for j in range(i):
                assert np.all(C[:, tri(i, j)] ** 2 <= C[:, tri(i, i)] * C[:, tri(j, j)] * (1 + 1e-5))


def test_p10_generator_truth(cfg1_tracks):
    tf, secs, out = cfg1_tracks
    ms = [sector_metrics(tf.label[s], out[s].order, out[s].hit_offset, out[s].hit_idx) for s in secs]
    m = summarize(ms)
    assert m["n_findable"] > 900
    assert m["efficiency"] >= 0.97 and m["fake_rate"] <= 0.05, m


def test_p10_config0_and_config4_truth(cfg0):
    out = run_timeframe(cfg0)
    m = summarize([sector_metrics(cfg0.label[0], out[0].order, out[0].hit_offset, out[0].hit_idx)])
    assert m["efficiency"] >= 0.95 and m["fake_rate"] <= 0.05, m
    tf4 = tpcsynth.generate(4, n_tracks=3000)
    secs = [0, 9, 20]
    out = run_timeframe(tf4, sectors=secs)
    m = summarize([sector_metrics(tf4.label[s], out[s].order, out[s].hit_offset, out[s].hit_idx) for s in secs])
    assert m["efficiency"] >= 0.85, m       # stress config: loopers, 10 % drop-out, 20 % noise


# ----------------------------------------------------------------------------------------
# P11 determinism, P12 z-translation
# ----------------------------------------------------------------------------------------
def _all_arrays(res):
    return [res.order, res.bin_start, res.link_up_raw, res.link_dn_raw, res.link_up, res.link_dn, res.start_hit,
            res.x_ref, res.par, res.cov, res.chi2, res.n_hits, res.n_fit, res.hit_offset, res.hit_idx]


def test_p11_determinism(cfg0):
    a = run_timeframe(cfg0)[0]
    b = run_timeframe(cfg0)[0]
    for u, v in zip(_all_arrays(a), _all_arrays(b)):
        assert np.array_equal(u, v)
    assert np.array_equal(a.z_ref, b.z_ref)


def test_p12_z_translation_is_exact():
    """A collision at t = 0 and the same collision shifted rigidly in z (time frame reading G9)
    give bit-identical links, hits, parameters and covariances; only z_ref shifts."""
    tf = tpcsynth.generate(1, n_tracks=500)
    s = 4
    y, row = tf.y[s], tf.row[s]
    zq = (np.round(tf.z[s].astype(np.float64) * 256.0) / 256.0).astype(np.float32)     # 2^-8 lattice
    shift = 4096.0 + 37.0 / 256.0
    P0 = tf.params
    P1 = P0.copy(grid_z_lo=float(np.float32(P0.grid_z_lo + shift)))
    assert float(np.float32(P0.grid_z_lo + shift)) == P0.grid_z_lo + shift
    z1 = (zq.astype(np.float64) + shift).astype(np.float32)
    assert np.array_equal(z1.astype(np.float64), zq.astype(np.float64) + shift)         # exact
    a = Oracle(P0).run(y, zq, row)
    b = Oracle(P1).run(y, z1, row)
    assert a.n_tracks > 50
    for u, v in zip(_all_arrays(a), _all_arrays(b)):
        assert np.array_equal(u, v)
    assert np.array_equal(a.z_ref + shift, b.z_ref)


# ----------------------------------------------------------------------------------------
# S5 decisions: hand-worked toy (tests/golden/toy_tracklets.txt)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("reverse_ids", [False, True])
def test_toy_tracklet_decisions(precision, reverse_ids):
    """Gap counting (phase B, phase C below the start row only), the phase-A gate from the third
    hit, tc_min_hits, window edges, search tie-breaks, the chi2 gate just inside / outside (threshold
    from the textbook prediction variance of a straight-line fit) and readings R2 / R3: expected
    membership written by hand in the golden file, never by an implementation."""
    import toy_tracklets
    scen = toy_tracklets.load()
    assert [s.name for s in scen] == ["A", "B", "C"] and sum(len(s.tracks) for s in scen) >= 20
    for sc in scen:
        y, z, row = sc.arrays(reverse_ids)
        res = Oracle(sc.params(), precision).run(y, z, row)
        toy_tracklets.check_result(sc, res, reverse_ids)


# ----------------------------------------------------------------------------------------
# full pipeline: tracks do not depend on the grid (bin size -> one bin per row = brute force)
# ----------------------------------------------------------------------------------------
def tracks_in_original_ids(res):
    """{original id of the start hit: (hit original ids, x_ref, z_ref, par, cov, chi2, n_fit)}"""
    o = res.order.astype(np.int64)
    out = {}
    for t in range(res.n_tracks):
        hits = o[res.hit_idx[res.hit_offset[t]:res.hit_offset[t + 1]]]
        out[int(o[res.trk_start_hit[t]])] = (tuple(hits.tolist()), res.x_ref[t], res.z_ref[t], tuple(res.par[t]),
                                             tuple(res.cov[t]), res.chi2[t], int(res.n_fit[t]))
    return out


@pytest.mark.parametrize("config,n_tracks,sector", [(1, 600, 3), (4, 1500, 0)])
def test_tracks_independent_of_grid_and_brute_force_search(config, n_tracks, sector):
    """P3 extended to S5: hit lists, parameters, covariances and chi2 in original-id space are
    bit-identical under other bin sizes / margins.  With bin_scale = 1000 every row is ONE bin, so
    the S2 windows and every S5 Search walk the whole row: the grid search equals brute force."""
    tf = tpcsynth.generate(config, n_tracks=n_tracks)
    y, z, row = tf.y[sector], tf.z[sector], tf.row[sector]
    assert y.shape[0] <= 8000
    sigma = tf.params.sigma
    base = tracks_in_original_ids(Oracle(tf.params).run(y, z, row))
    assert len(base) > 60
    for bs, gm in ((0.5, 0.01), (1.7, 0.01), (3.0, 0.5), (1000.0, 0.0)):
        P2 = tpcsynth.default_params(n_sectors=36, sigma=sigma, bin_scale=bs, grid_margin=gm)
        if bs == 1000.0:
            assert np.all(P2.grid_ny == 1) and np.all(P2.grid_nz == 1)
        got = tracks_in_original_ids(Oracle(P2).run(y, z, row))
        assert got == base, (bs, gm)


def test_search_on_dense_rows_equals_whole_row_scan():
    """Dense uniform clusters (several candidates in every search window, S5 decisions dominated by
    Search): one bin per row (whole-row scan) and the default grid give bit-identical tracks."""
    P = tpcsynth.default_params(n_sectors=1)
    rng = np.random.default_rng(8)
    n = 1800
    row = rng.integers(0, 40, n).astype(np.uint16)
    y = (rng.random(n) * 10.0 - 5.0).astype(np.float32)
    z = (rng.random(n) * 24.0).astype(np.float32)
    # thread a few straight tracks through the noise so that searches have something to extend
    rx = P.row_x.astype(np.float64)
    r2, y2, z2, _ = tpcsynth.straight_tracks(rx[:40], [-3.0, 0.0, 2.5], [0.05, -0.02, 0.0], [4.0, 12.0, 20.0], [0.1, 0.0, -0.1])
    row = np.concatenate([row, r2]); y = np.concatenate([y, y2.astype(np.float32)]); z = np.concatenate([z, z2.astype(np.float32)])
    P1 = tpcsynth.default_params(n_sectors=1, bin_scale=1000.0, grid_margin=0.0)
    a = tracks_in_original_ids(Oracle(P).run(y, z, row))
    b = tracks_in_original_ids(Oracle(P1).run(y, z, row))
    assert len(a) >= 3 and a == b


# ----------------------------------------------------------------------------------------
# n14 (d z / d q/pT) where its second term, (k d) d^2 / 12, dominates
# ----------------------------------------------------------------------------------------
def test_jacobian_n14_arc_term():
    """A long symmetric step (sin phi: -a -> +a, so dy = 0 and the chord term (dy/d) j4 of n14
    vanishes) leaves n14 = p3 Bc (k d) d^2 c12.  Compared with central differences of the z
    transport in q/pT: pins c12 = 1/12 (1/6 would be off by a factor 2)."""
    P = tpcsynth.default_params(n_sectors=1)
    orc = Oracle(P, "f64")
    Bc = float(P.kappa_per_qpt)
    x1, x2 = 100.0, 130.0
    p4 = 5.0
    a = 0.5 * p4 * Bc * (x2 - x1)
    p = np.array([1.0, 2.0, -a, 0.8, p4])
    tri = lambda i, j: i * (i + 1) // 2 + j

    def z_at(q4):
        q = p.copy(); q[4] = q4
        ok, s = orc.kf_propagate(_state(x1, q), x2)
        assert ok
        return s[2], s[1]
    z0, y_end = z_at(p4)
    assert abs(y_end - 1.0) < 1e-12                                   # symmetric step: dy == 0
    h = 1e-4
    fd = (z_at(p4 + h)[0] - z_at(p4 - h)[0]) / (2 * h)
    C = np.zeros(15); C[tri(4, 4)] = 1.0
    ok, s = orc.kf_propagate(_state(x1, p, C), x2)
    n14 = s[6 + tri(4, 1)]                                            # C'_41 = J_14 * J_44
    want = p[3] * Bc * (p4 * Bc * 30.0) * 900.0 / 12.0                # p3 Bc (k d) d^2 / 12 with d = dx
    assert abs(fd - want) < 0.02 * want and abs(n14 - fd) < 0.02 * abs(fd), (n14, fd, want)


# ----------------------------------------------------------------------------------------
# S6 tracklet selector
# ----------------------------------------------------------------------------------------
def _read_selector_toy():
    import os
    tracks, exp = [], {}
    owner = n_own = None
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "toy_selector.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        head, _, body = line.partition(":")
        vals = [int(v) for v in body.split()]
        if head.startswith("track"):
            tracks.append(vals)
        elif head == "owner":
            owner = vals
        elif head == "n_own":
            n_own = vals
        else:
            exp[int(head.split()[1])] = vals
    return tracks, owner, n_own, exp


def test_selector_toy_worked_example():
    from oracle import select_tracks
    tracks, owner, n_own, exp = _read_selector_toy()
    off = np.concatenate([[0], np.cumsum([len(t) for t in tracks])])
    idx = np.concatenate(tracks)
    for permille, want in exp.items():
        o, w, s = select_tracks(len(owner), off, idx, permille)
        assert o.tolist() == owner and w.tolist() == n_own and s.tolist() == want, permille


def numpy_selector(n_clusters, hit_offset, hit_idx, permille):
    """Independent formulation: sort all (cluster, -n_hits, track) triples; the first of every cluster owns it."""
    nt = len(hit_offset) - 1
    nh = np.diff(hit_offset).astype(np.int64)
    trk = np.repeat(np.arange(nt), nh)
    order = np.lexsort((trk, -nh[trk], hit_idx))
    c_sorted = hit_idx[order]
    first = np.ones(len(order), bool); first[1:] = c_sorted[1:] != c_sorted[:-1]
    owner = np.full(n_clusters, -1, np.int64)
    owner[c_sorted[first]] = trk[order][first]
    n_own = np.bincount(trk[owner[hit_idx] == trk], minlength=nt)
    sel = np.nonzero((nh - n_own) * 1000 <= permille * nh)[0]
    return owner, n_own, sel


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_selector_equals_sort_formulation(seed):
    from oracle import select_tracks
    rng = np.random.default_rng(seed)
    n, nt = 400, 120
    lists = []
    for t in range(nt):
        k = int(rng.integers(1, 30))
        base = int(rng.integers(0, n - 40))
        lists.append(np.sort(rng.choice(np.arange(base, base + 40), size=k, replace=False)))   # overlapping neighbourhoods
    off = np.concatenate([[0], np.cumsum([len(l) for l in lists])]).astype(np.int32)
    idx = np.concatenate(lists).astype(np.int32)
    for permille in (0, 250, 500, 900):
        o, w, s = select_tracks(n, off, idx, permille)
        o2, w2, s2 = numpy_selector(n, off, idx, permille)
        assert np.array_equal(o, o2) and np.array_equal(w, w2) and np.array_equal(s, s2)
        covered = np.zeros(n, bool); covered[idx] = True
        assert np.array_equal(o >= 0, covered) and w.sum() == covered.sum()       # every covered cluster has one owner


def test_selector_removes_clones_and_keeps_efficiency(cfg1_tracks):
    """Generator truth (P10) before and after S6 on config-1 kinematics: about four clones per particle
    (reading N3) fall to about one, the efficiency is unchanged, fakes do not grow."""
    tf, secs, _ = cfg1_tracks
    orc = Oracle(tf.params)
    before, after = [], []
    for s in secs:
        r = orc.run(tf.y[s], tf.z[s], tf.row[s], stage_mask=0x3F)
        assert r.selected.shape[0] > 0 and np.all(np.diff(r.selected) > 0)
        before.append(sector_metrics(tf.label[s], r.order, r.hit_offset, r.hit_idx))
        off = np.concatenate([[0], np.cumsum(r.n_hits[r.selected])]).astype(np.int32)
        idx = np.concatenate([r.hit_idx[r.hit_offset[t]:r.hit_offset[t + 1]] for t in r.selected])
        after.append(sector_metrics(tf.label[s], r.order, off, idx))
    b, a = summarize(before), summarize(after)
    assert b["clone_rate"] > 0.6, b                       # >= 2.5 found tracks per matched particle
    assert a["clone_rate"] < 0.05, a
    assert a["efficiency"] >= b["efficiency"] - 0.005 and a["efficiency"] >= 0.97, (a, b)
    assert a["fake_rate"] <= b["fake_rate"] + 0.01, (a, b)


# ----------------------------------------------------------------------------------------
# S7 track-residual front end
# ----------------------------------------------------------------------------------------
def test_residuals_vanish_on_exact_helices():
    """Noise-free helices (P6 fixture, double): every cluster is owned by its track and its residual to the
    fitted helix is zero to 2e-5 cm (the fit itself recovers the helix to 1e-5 relative, P6); the quantised
    residuals are all 0."""
    P = tpcsynth.default_params(n_sectors=1)
    y, z, row, lab = _helix_sector(P, HELIX_TRACKS, np.float64)
    res = Oracle(P, "f64").run(y, z, row, stage_mask=0x7F)
    assert res.n_tracks == len(HELIX_TRACKS) and len(res.selected) == len(HELIX_TRACKS)
    assert np.all(res.res_trk >= 0)
    assert np.abs(res.res_y).max() < 2e-5 and np.abs(res.res_z).max() < 2e-5
    assert not res.q_y.any() and not res.q_z.any()


def test_residuals_equal_closed_form_circle(cfg0):
    """Residual of every attached cluster vs the closed-form helix through the fitted state (x_ref, par):
    sin phi(x) = sin phi0 + kappa (x - x0); y(x) = y0 + (cos phi0 - cos phi(x)) / kappa;
    z(x) = z0 + dz/ds * (phi(x) - phi0) / kappa -- circle geometry with asin, independent of the oracle's
    hit-to-hit chord transport.  Pins which state is transported, the walk, the signs and K-rule Z."""
    tf = cfg0
    P = tf.params
    res = Oracle(P, "f64").run(tf.y[0], tf.z[0], tf.row[0], stage_mask=0x7F)
    Bc = float(P.kappa_per_qpt)
    rx = P.row_x.astype(np.float64)
    srow = tf.row[0][res.order].astype(np.int64)
    m = np.nonzero(res.res_trk >= 0)[0]
    assert m.size > 3000
    t = res.res_trk[m]
    assert np.all(np.isin(t, res.selected)) and np.array_equal(res.owner[m], t)
    x0 = res.x_ref[t]; p = res.par[t]
    kappa = p[:, 4] * Bc
    sp = p[:, 2] + kappa * (rx[srow[m]] - x0)
    ok = np.abs(kappa) > 1e-9
    yh = np.where(ok, p[:, 0] + (np.sqrt(1 - p[:, 2] ** 2) - np.sqrt(1 - sp ** 2)) / np.where(ok, kappa, 1.0), np.nan)
    zh = np.where(ok, p[:, 1] + p[:, 3] * (np.arcsin(sp) - np.arcsin(p[:, 2])) / np.where(ok, kappa, 1.0), np.nan)
    assert ok.mean() > 0.99
    assert np.nanmax(np.abs(res.res_y[m] - (res.sy[m] - yh))) < 1e-7
    assert np.nanmax(np.abs(res.res_z[m] - ((res.sz[m] - res.z_ref[t]) - zh))) < 1e-6
    # every cluster a selected track owns is attached (no transport failed on this input)
    owned = np.isin(res.owner, res.selected) & (res.owner >= 0)
    assert np.array_equal(owned, res.res_trk >= 0)


def test_residual_statistics_and_quantiser(cfg1_tracks):
    """fp32, config-1 kinematics: residuals of attached clusters are centred with the cluster resolution
    (sigma = 0.1 cm, slightly less: the fit absorbs part of it); q = rint(res * 128) with numpy's round-half-even."""
    tf, secs, _ = cfg1_tracks
    orc = Oracle(tf.params)
    ry, rz = [], []
    for s in secs[:3]:
        r = orc.run(tf.y[s], tf.z[s], tf.row[s], stage_mask=0x7F)
        m = r.res_trk >= 0
        assert m.mean() > 0.85                                   # most clusters are attached to a selected track
        f32 = np.float32
        assert np.array_equal(r.q_y[m], np.clip(np.rint(r.res_y[m].astype(f32) * f32(128.0)), -32767, 32767).astype(np.int16))
        assert np.array_equal(r.q_z[m], np.clip(np.rint(r.res_z[m].astype(f32) * f32(128.0)), -32767, 32767).astype(np.int16))
        assert not r.q_y[~m].any() and not r.res_y[~m].any()
        lab = tf.label[s][r.order]
        good = m & (lab >= 0)
        ry.append(r.res_y[good]); rz.append(r.res_z[good])
    ry = np.concatenate(ry); rz = np.concatenate(rz)
    core_y = ry[np.abs(ry) < 0.5]; core_z = rz[np.abs(rz) < 0.5]
    assert core_y.size > 0.98 * ry.size
    assert abs(core_y.mean()) < 0.003 and abs(core_z.mean()) < 0.003
    assert 0.085 < core_y.std() < 0.105 and 0.085 < core_z.std() < 0.105


# ----------------------------------------------------------------------------------------
# S8 cross-sector merging + refit
# ----------------------------------------------------------------------------------------
def test_rotate_follows_exact_circle_geometry():
    """Rotate + Propagate vs the generator's exact circle geometry (tpcsynth.truth_state: double precision,
    atan2 / sinh, the same helix expressed in the local frames of two neighbouring sectors)."""
    tf = tpcsynth.generate(1, n_tracks=400)
    P = tf.params
    orc = Oracle(P, "f64")
    rx = P.row_x.astype(np.float64)
    ca, sa = math.cos(math.pi / 9), math.sin(math.pi / 9)
    n_ok = 0
    for trk in range(tf.trk_pt.shape[0]):
        if tf.trk_pt[trk] < 0.4:
            continue
        for s in range(0, 36, 3):
            for x in (rx[10], rx[40], rx[75], rx[110], rx[140]):
                a = tpcsynth.truth_state(tf, trk, s, float(x))
                if a is None or not (0.165 * x <= abs(a["y"]) <= 0.19 * x) or abs(a["sinphi"]) > 0.6:   # at the edge of sector s
                    continue
                up = a["y"] > 0                                                     # leaves towards s+1 (y > 0) or s-1
                n_sec = (s // 18) * 18 + ((s % 18) + (1 if up else 17)) % 18
                st = _state(x, [a["y"], a["z"], a["sinphi"], a["dzds"], a["p4"]])
                ok, r = orc.kf_rotate(st, ca, sa if up else -sa)
                assert ok
                x2 = float(rx[np.argmin(np.abs(rx - r[0]))])                        # nearest pad row of the neighbour
                b = tpcsynth.truth_state(tf, trk, n_sec, x2)
                if b is None or abs(b["sinphi"]) > 0.9:
                    continue
                ok, q = orc.kf_propagate(r, x2)
                assert ok
                assert abs(q[1] - b["y"]) < 1e-8 and abs(q[3] - b["sinphi"]) < 1e-10, (trk, s, q[1], b["y"])
                assert abs(q[2] - b["z"]) < 1e-6 and q[4] == a["dzds"] and q[5] == a["p4"]
                n_ok += 1
    assert n_ok > 25


def test_rotate_covariance_jacobian_finite_differences():
    """C' = J C J^T of Rotate vs central differences of (rotate, then back onto the unperturbed plane)."""
    P = tpcsynth.default_params(n_sectors=1)
    orc = Oracle(P, "f64")
    ca, sa = math.cos(math.pi / 9), -math.sin(math.pi / 9)
    x = 150.0
    p = np.array([24.0, -3.0, 0.35, 0.6, -2.0])
    ok, base = orc.kf_rotate(_state(x, p), ca, sa)
    assert ok
    x_new = base[0]

    def image(q):
        ok, r = orc.kf_rotate(_state(x, q), ca, sa)
        assert ok
        ok, r = orc.kf_propagate(r, x_new)           # the perturbed point lies on another plane: bring it back
        assert ok
        return r[1:6]
    tri = lambda i, j: i * (i + 1) // 2 + j
    J_fd = np.zeros((5, 5))
    for j in range(5):
        h = 1e-6
        dp = np.zeros(5); dp[j] = h
        J_fd[:, j] = (image(p + dp) - image(p - dp)) / (2 * h)
    # J from the covariance transform: for C = e_j e_j^T + e_k e_k^T ... use single-entry covariances
    J = np.zeros((5, 5))
    for j in range(5):
        C = np.zeros(15); C[tri(j, j)] = 1.0
        ok, r = orc.kf_rotate(_state(x, p, C), ca, sa)
        Cn = r[6:21]
        d = np.array([Cn[tri(i, i)] for i in range(5)])          # J[i,j]^2
        jj = int(np.argmax(d))
        col = np.array([Cn[tri(max(i, jj), min(i, jj))] for i in range(5)]) / math.sqrt(d[jj])
        if col @ J_fd[:, j] < 0:
            col = -col
        J[:, j] = col
    assert np.allclose(J, J_fd, rtol=1e-6, atol=1e-7), (J, J_fd)
    assert abs(J[0, 0] - 1) > 0.05 and abs(J[2, 0]) > 1e-4 and abs(J[1, 0]) > 0.05      # the non-trivial terms are exercised


@pytest.fixture(scope="module")
def merged_cfg1():
    from oracle import run_timeframe_merged
    tf = tpcsynth.generate(1, n_tracks=4000)
    res, mg = run_timeframe_merged(tf)
    return tf, res, mg


def _selected_majority(tf, res, s):
    from tpcsynth.truth import match_tracks
    r = res[s]
    lab = tf.label[s][r.order]
    off = np.concatenate([[0], np.cumsum(r.n_hits[r.selected])]).astype(np.int32)
    idx = (np.concatenate([r.hit_idx[r.hit_offset[t]:r.hit_offset[t + 1]] for t in r.selected]) if len(r.selected)
           else np.empty(0, np.int32))
    return match_tracks(lab, off, idx)[0]


def test_merge_links_invariants_and_truth(merged_cfg1):
    tf, res, mg = merged_cfg1
    maj = [_selected_majority(tf, res, s) for s in range(36)]
    n_links = good = 0
    gaps = []
    for s in range(36):
        m, r = mg[s], res[s]
        for ia in np.nonzero(m.next_sec >= 0)[0]:
            ns_, ib = int(m.next_sec[ia]), int(m.next_trk[ia])
            # neighbours on the same side; links are mutual; the upper segment starts 1..8 rows above the lower one
            assert ns_ // 18 == s // 18 and (ns_ % 18 - s % 18) % 18 in (1, 17)
            assert mg[ns_].prev_sec[ib] == s and mg[ns_].prev_trk[ib] == ia
            gap = res[ns_].first_row[res[ns_].selected[ib]] - r.last_row[r.selected[ia]]
            assert 1 <= gap <= 8
            gaps.append(gap)
            n_links += 1
            good += int(maj[s][ia] >= 0 and maj[s][ia] == maj[ns_][ib])
        assert (m.prev_sec >= 0).sum() == sum(int((mg[t].next_sec == s).sum()) for t in range(36))
    assert n_links > 3000 and good >= 0.99 * n_links, (n_links, good)
    assert min(gaps) == 1 and max(gaps) >= 4
    # efficiency: pairs of selected tracks of neighbouring sectors with the same particle, consecutive in row
    # (upper starts 1..8 rows above the lower one's end), are linked
    want = have = 0
    for s in range(36):
        r = res[s]
        for d in (1, 17):
            t = (s // 18) * 18 + (s % 18 + d) % 18
            rt = res[t]
            by_label = {}
            for ib, lb in enumerate(maj[t]):
                if lb >= 0:
                    by_label.setdefault(int(lb), []).append(ib)
            for ia, la in enumerate(maj[s]):
                for ib in by_label.get(int(la), []) if la >= 0 else []:
                    gap = rt.first_row[rt.selected[ib]] - r.last_row[r.selected[ia]]
                    if 1 <= gap <= 8:
                        want += 1
                        have += int(mg[s].next_sec[ia] == t and mg[s].next_trk[ia] == ib)
    assert want > 3000 and have >= 0.93 * want, (want, have)


def test_merged_refit_statistics(merged_cfg1):
    """The refit over the union of the segments: unit pulls against generator truth at the reference plane of the
    lowest segment, chi2 / ndf = 1, every hit of every segment fitted, covariance smaller than the head's own."""
    tf, res, mg = merged_cfg1
    maj = [_selected_majority(tf, res, s) for s in range(36)]
    pulls, red, shrink = [], [], []
    tri = lambda i: i * (i + 1) // 2 + i
    n_chain = 0
    for s in range(36):
        m, r = mg[s], res[s]
        for k in range(len(m.head)):
            segs = list(zip(m.seg_sec[m.seg_offset[k]:m.seg_offset[k + 1]], m.seg_trk[m.seg_offset[k]:m.seg_offset[k + 1]]))
            assert segs[0] == (s, m.head[k]) and len(segs) == m.n_seg[k] >= 2
            tot = sum(int(res[a].n_hits[res[a].selected[b]]) for a, b in segs)
            n_chain += 1
            if m.n_fit[k] != tot:
                continue                                        # a transport failed on the way down (rare)
            assert m.frame_seg[k] == 0 and m.n_hits[k] == tot
            t_head = r.selected[m.head[k]]
            assert m.x_ref[k] == r.x_ref[t_head] and m.z_ref[k] == r.z_ref[t_head]
            labs = {int(maj[a][b]) for a, b in segs}
            if len(labs) != 1 or -1 in labs or tot < 60:
                continue
            tr = tpcsynth.truth_state(tf, labs.pop(), s, float(m.x_ref[k]))
            if tr is None:
                continue
            got = np.array([m.par[k, 0], m.z_ref[k] + m.par[k, 1], m.par[k, 2], m.par[k, 3], m.par[k, 4]])
            want = np.array([tr["y"], tr["z"], tr["sinphi"], tr["dzds"], tr["p4"]])
            err = np.sqrt(np.array([m.cov[k][tri(i)] for i in range(5)]))
            pulls.append((got - want) / err)
            red.append(m.chi2[k] / (2 * m.n_fit[k] - 5))
            shrink.append(m.cov[k][tri(4)] / r.cov[t_head][tri(4)])
    pulls = np.array(pulls)
    assert n_chain > 1500 and pulls.shape[0] > 800
    core = np.all(np.abs(pulls) < 5, axis=1)
    assert core.mean() > 0.95
    pc = pulls[core]
    assert np.all(np.abs(pc.mean(axis=0)) < 0.12), pc.mean(axis=0)
    assert np.all(np.abs(pc.std(axis=0) - 1.0) < 0.12), pc.std(axis=0)
    assert abs(np.mean(np.array(red)[core]) - 1.0) < 0.06
    assert np.median(shrink) < 0.5                              # the longer lever arm pins q/pT down


def test_merge_row_gap_bounds_are_inclusive():
    """mg_max_row_gap is data: with 2, links with a gap of exactly 2 rows exist and none is larger (pins `1 <= gap <= max`)."""
    from oracle import run_timeframe_merged
    tf = tpcsynth.generate(1, n_tracks=2500)
    tf.params = tf.params.copy(mg_max_row_gap=2)
    res, mg = run_timeframe_merged(tf)
    gaps = []
    for s in range(36):
        for ia in np.nonzero(mg[s].next_sec >= 0)[0]:
            b = res[mg[s].next_sec[ia]]
            gaps.append(int(b.first_row[b.selected[mg[s].next_trk[ia]]] - res[s].last_row[res[s].selected[ia]]))
    assert len(gaps) > 300 and min(gaps) == 1 and max(gaps) == 2 and gaps.count(2) > 20


def test_merge_toy_worked_example():
    """S8 match decisions on hand-made tracks (tests/golden/toy_merge.txt): inclusive window edges, row-gap bounds,
    the z pre-cut, mutual best without fall-back, ties by (sector, track), chains through three sectors."""
    import os
    from oracle import merge_links_of_tables
    P = tpcsynth.default_params(n_sectors=6, row_x=64.0 + np.arange(32), sigma=0.125)
    P = P.copy(sectors_per_side=3, sector_cos=1.0, sector_sin=0.0, mg_max_row_gap=8, mg_dy=1.0, mg_dz=1.0, mg_dsin=0.0625,
               mg_zpre=32.0)
    sectors = [[] for _ in range(6)]
    where, links = {}, []
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "toy_merge.txt")):
        f = line.split("#")[0].split()
        if not f:
            continue
        if f[0] == "link":
            links.append((f[1], f[2]))
            continue
        kind, name, s = f[0], f[1], int(f[2])
        if kind == "lower":
            last, y, zref = int(f[3]), float(f[4]), float(f[5])
            noout = "noout" in f
            p3 = float(f[6]) if len(f) > 6 and f[6] != "noout" else 0.0
            t = dict(first_row=0, last_row=last, x_ref=64.0, z_ref=zref, par=[y, 0.0, 0.0, p3, 0.0],
                     out=None if noout else [64.0 + last, y, 0.0, 0.0, p3, 0.0])
        elif kind == "upper":
            first, y, zref = int(f[3]), float(f[4]), float(f[5])
            p1 = float(f[6]) if len(f) > 6 else 0.0
            sp = float(f[7]) if len(f) > 7 else 0.0
            t = dict(first_row=first, last_row=31, x_ref=64.0 + first, z_ref=zref, par=[y, p1, sp, 0.0, 0.0], out=None)
        else:   # mid: first_row last_row y z_ref -- both an upper and a lower segment
            first, last, y, zref = int(f[3]), int(f[4]), float(f[5]), float(f[6])
            t = dict(first_row=first, last_row=last, x_ref=64.0 + first, z_ref=zref, par=[y, 0.0, 0.0, 0.0, 0.0],
                     out=[64.0 + last, y, 0.0, 0.0, 0.0, 0.0])
        where[name] = (s, len(sectors[s]))
        sectors[s].append(t)
    assert len(links) == 13 and len(where) == 42
    for precision in ("f32", "f64"):
        got = merge_links_of_tables(P, sectors, precision)
        want = [([-1] * len(t), [-1] * len(t), [-1] * len(t), [-1] * len(t)) for t in sectors]
        for lo, up in links:
            (sa, ia), (sb, ib) = where[lo], where[up]
            want[sa][0][ia] = sb; want[sa][1][ia] = ib; want[sb][2][ib] = sa; want[sb][3][ib] = ia
        for s in range(6):
            assert got[s] == tuple(want[s]), (precision, s, got[s], want[s])
