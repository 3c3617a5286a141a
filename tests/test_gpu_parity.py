"""Parity of the CUDA path (through the C-ABI) against the CPU oracle, element by element.

Run on the B200 box: python -m pytest tests -m gpu.  Inputs are the seeded synthetic generators of
tpcsynth (BASELINE.json:7-11 recipes), never values produced by the CUDA path.
"""
import os

import numpy as np
import pytest

import tpcsynth
from oracle import Oracle
from parity import ParityError, compare_sector, compare_timeframe

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    import paper_2208_07412_b200 as p
    p.load_library()
    return p


#: TPCCA_TEST_WS_FILL=0xff (or 0x7f, ...) poisons every workspace before tpcca_create: the stand-in for
#: `compute-sanitizer --tool initcheck`, which is closed on this GPU pool (profiles/r2_sanitizers.md)
WS_FILL = int(os.environ["TPCCA_TEST_WS_FILL"], 0) if os.environ.get("TPCCA_TEST_WS_FILL") else None


def run_gpu(pkg, tf, stages=0x1F, max_start_hits=0):
    n = max(tf.n_clusters, 1)
    trk = pkg.Tracker(tf.params, max_clusters=n, max_start_hits=max_start_hits, workspace_fill=WS_FILL)
    trk.load_timeframe(tf)
    trk.run(stages)
    trk.sync()
    return trk


class ArrTF:
    """Minimal time-frame-like holder for hand-made inputs."""
    def __init__(self, params, secs):
        self.params = params
        self.y = [np.asarray(s[0], np.float32) for s in secs]
        self.z = [np.asarray(s[1], np.float32) for s in secs]
        self.row = [np.asarray(s[2], np.uint16) for s in secs]
        self.x = [params.row_x[r] for r in self.row]
        self.q = [np.ones(len(r), np.float32) for r in self.row]

    @property
    def n_sectors(self):
        return len(self.y)

    @property
    def n_clusters(self):
        return int(sum(len(a) for a in self.y))


def check(pkg, tf, stages=0x1F, sectors=None, **kw):
    trk = run_gpu(pkg, tf, stages, **kw)
    orc = Oracle(tf.params)
    rep = compare_timeframe(trk, tf, orc, sectors=sectors, stages=stages)
    trk.close()
    return rep


# ------------------------------------------------------------------------------------------------
def test_config0_full_pipeline(pkg, cfg0):
    rep = check(pkg, cfg0)
    assert rep["n_tracks"] > 100 and rep["links_differing"] == 0


def test_config1_small_36_sectors(pkg, cfg1_small):
    rep = check(pkg, cfg1_small)
    assert rep["sectors"] == 36 and rep["n_tracks"] > 1000 and rep["links_differing"] == 0


def test_config4_small_stress(pkg):
    tf = tpcsynth.generate(4, n_tracks=1500)
    rep = check(pkg, tf)
    assert rep["n_tracks"] > 500 and rep["links_differing"] == 0


def test_timeframe_slice_small(pkg):
    """Config-2 recipe at 2 orbits: several collisions shifted along z (reading G9)."""
    tf = tpcsynth.generate(2, n_orbits=2, mult_scale=0.3)
    assert tf.coll_t.shape[0] >= 3
    rep = check(pkg, tf)
    assert rep["n_tracks"] > 300 and rep["links_differing"] == 0


def test_timeframe_slice_dense(pkg):
    """One orbit of the time-frame recipe at 2.75x multiplicity: the occupancy of the ~4e8-cluster footprint
    BASELINE.json:10 names (dense windows: S2 medium / slow paths, long candidate lists in the S5 search)."""
    tf = tpcsynth.generate(2, n_orbits=1, mult_scale=2.75, seed=220807499)
    assert tf.n_clusters > 200_000
    rep = check(pkg, tf)
    assert rep["n_tracks"] > 2000 and rep["links_differing"] == 0


def test_stage_by_stage_equals_all_at_once(pkg, cfg0):
    tf = cfg0
    a = run_gpu(pkg, tf, 0x1F)
    b = pkg.Tracker(tf.params, max_clusters=tf.n_clusters)
    b.load_timeframe(tf)
    for m in (1, 2, 4, 8, 16):
        b.run(m)
    b.sync()
    ga, gb = a.get_tracks(0), b.get_tracks(0)
    for f in ("order", "sy", "sz", "bin_start", "row_start", "link_up_raw", "link_dn_raw", "link_up", "link_dn",
              "start_hit", "par", "cov", "chi2", "hit_offset", "hit_idx", "trk_start_hit"):
        assert np.array_equal(getattr(ga, f), getattr(gb, f)), f
    # partial masks are compared with the oracle as well
    orc = Oracle(tf.params)
    for m in (1, 3, 7, 15):
        c = run_gpu(pkg, tf, m)
        compare_timeframe(c, tf, orc, stages=m)
        c.close()
    a.close(); b.close()


def test_determinism_and_context_reuse(pkg, cfg1_small):
    """P11: same input twice -> byte-identical outputs; a context is reusable after reset."""
    tf = cfg1_small
    trk = run_gpu(pkg, tf)
    first = [trk.get_tracks(s) for s in (0, 5, 20)]
    trk.load_timeframe(tf)      # reset + reload
    trk.run()
    second = [trk.get_tracks(s) for s in (0, 5, 20)]
    for a, b in zip(first, second):
        for f in ("order", "bin_start", "link_up_raw", "link_dn", "start_hit", "par", "cov", "chi2", "hit_idx"):
            assert np.array_equal(getattr(a, f), getattr(b, f)), f
    trk.close()


def test_empty_and_tiny_inputs(pkg):
    P = tpcsynth.default_params(n_sectors=3)
    e = (np.empty(0, np.float32), np.empty(0, np.float32), np.empty(0, np.uint16))
    # all empty
    rep = check(pkg, ArrTF(P, [e, e, e]))
    assert rep["n_tracks"] == 0
    # one cluster; a sector in the middle empty; clusters outside the grid (reading N9)
    one = (np.array([0.5], np.float32), np.array([10.0], np.float32), np.array([7], np.uint16))
    out = (np.array([-1e3, 1e3, 0.0, 0.0], np.float32), np.array([10.0, 10.0, -50.0, 1e6], np.float32),
           np.array([5, 5, 5, 5], np.uint16))
    check(pkg, ArrTF(P, [one, e, out]))
    # rows 0 and n_rows-1 only
    edge = (np.zeros(6, np.float32), np.arange(6, dtype=np.float32), np.array([0, 0, 151, 151, 0, 151], np.uint16))
    check(pkg, ArrTF(P, [edge, one, e]))


def test_ties_and_duplicates(pkg):
    """Reading N7: duplicated clusters; ties go to the smallest original id (needs order[] on the GPU)."""
    P = tpcsynth.default_params(n_sectors=1)
    y = np.array([0.0, 0.5, -0.5, 0.5, -0.5], np.float32)
    z = np.array([10.0, 10.5, 9.5, 10.5, 9.5], np.float32)
    row = np.array([10, 11, 9, 11, 9], np.uint16)
    check(pkg, ArrTF(P, [(y, z, row)]))
    # many exact duplicates on three rows, shuffled ids
    rng = np.random.default_rng(3)
    yy = np.repeat(np.array([0.0, 0.25, 0.5], np.float32), 40)
    zz = np.repeat(np.array([20.0, 20.5, 21.0], np.float32), 40)
    rr = np.repeat(np.array([20, 21, 22], np.uint16), 40)
    p = rng.permutation(120)
    check(pkg, ArrTF(P, [(yy[p], zz[p], rr[p])]))


@pytest.mark.parametrize("seed,n,zmax", [(1, 2000, 30.0), (2, 6000, 12.0)])
def test_dense_random_windows(pkg, seed, n, zmax):
    """Dense uniform clusters: many candidates per window (overflows the shared-memory candidate
    cache at the denser setting), many occupied bins, S5 searches with several candidates."""
    P = tpcsynth.default_params(n_sectors=1)
    rng = np.random.default_rng(seed)
    row = rng.integers(0, 12, n).astype(np.uint16)
    y = (rng.random(n) * 16.0 - 8.0).astype(np.float32)
    z = (rng.random(n) * zmax).astype(np.float32)
    check(pkg, ArrTF(P, [(y, z, row)]))


def test_oversized_buckets_and_tiles(pkg):
    """Thousands of clusters in a few rows and a short z range: S1 coarse buckets beyond the shared-memory
    sort (global-memory bucket path), S2 tiles whose neighbour runs exceed the staging buffer (global path),
    bins holding many clusters with shuffled ids."""
    P = tpcsynth.default_params(n_sectors=2)
    rng = np.random.default_rng(11)
    n = 9000
    row = rng.integers(4, 8, n).astype(np.uint16)
    y = (rng.random(n) * 30.0 - 15.0).astype(np.float32)
    z = (rng.random(n) * 120.0).astype(np.float32)
    e = (np.empty(0, np.float32), np.empty(0, np.float32), np.empty(0, np.uint16))
    check(pkg, ArrTF(P, [(y, z, row), e]))
    check(pkg, ArrTF(P, [e, (y[:3000], z[:3000] * 0.02, row[:3000])]))


def test_grid_variants(pkg):
    """P3 on the GPU: other bin sizes / margins (bin ranges spanning more than 3 bins)."""
    tf = tpcsynth.generate(1, n_tracks=600)
    for bs, gm in ((0.5, 0.01), (1.7, 0.01), (3.0, 0.5)):
        P2 = tpcsynth.default_params(n_sectors=2, bin_scale=bs, grid_margin=gm)
        check(pkg, ArrTF(P2, [(tf.y[s], tf.z[s], tf.row[s]) for s in (3, 4)]))


def test_toy_worked_example(pkg):
    path = os.path.join(os.path.dirname(__file__), "golden", "toy_links.txt")
    rows, ys, zs, exp = [], [], [], []
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
        exp.append([int(v) for v in f[4:8]])
    exp = np.array(exp)
    P = tpcsynth.default_params(n_sectors=1, row_x=64.0 + 1.0 * np.arange(8), sigma=0.125)
    tf = ArrTF(P, [(ys, zs, rows)])
    trk = run_gpu(pkg, tf, 0xF)
    g = trk.get_tracks(0)
    o = g.order.astype(np.int64)

    def to_orig(a):
        out = np.full(g.n, -1, np.int64)
        m = a >= 0
        out[o[m]] = o[a[m]]
        return out
    assert to_orig(g.link_up_raw).tolist() == exp[:, 0].tolist()
    assert to_orig(g.link_dn_raw).tolist() == exp[:, 1].tolist()
    assert to_orig(g.link_up).tolist() == exp[:, 2].tolist()
    assert to_orig(g.link_dn).tolist() == exp[:, 3].tolist()
    assert sorted(o[g.start_hit].tolist()) == sorted(exp_start)
    trk.close()


@pytest.mark.parametrize("reverse_ids", [False, True])
def test_toy_tracklet_decisions(pkg, reverse_ids):
    """The hand-worked S5 decision toy (tests/golden/toy_tracklets.txt) through the CUDA path: expected
    membership written by hand (gaps, phase-A gate, min hits, window edges, tie-breaks, chi2 gate, R2 / R3)."""
    import toy_tracklets
    for sc in toy_tracklets.load():
        y, z, row = sc.arrays(reverse_ids)
        tf = ArrTF(sc.params(), [(y, z, row)])
        trk = run_gpu(pkg, tf)
        toy_tracklets.check_result(sc, trk.get_tracks(0), reverse_ids)
        compare_timeframe(trk, tf, Oracle(tf.params))
        trk.close()


def test_straight_tracks_dyadic(pkg):
    """P4 on the GPU: exact recovery, 152-hit tracks, rows 0 and 151 attached by the search."""
    row_x = 64.0 + 0.75 * np.arange(152)
    P = tpcsynth.default_params(n_sectors=1, row_x=row_x)
    nt = 12
    row, y, z, trk_id = tpcsynth.straight_tracks(row_x, -6.0 + np.arange(nt), (np.arange(nt) - 6) / 64.0,
                                                 8.0 + 16.0 * np.arange(nt), (np.arange(nt) - 4) / 8.0)
    perm = np.random.default_rng(5).permutation(row.shape[0])
    tf = ArrTF(P, [(y[perm], z[perm], row[perm])])
    trk = run_gpu(pkg, tf)
    g = trk.get_tracks(0)
    assert g.n_tracks == nt and np.all(g.n_hits == 152) and np.all(g.first_row == 0) and np.all(g.last_row == 151)
    compare_timeframe(trk, tf, Oracle(P))
    trk.close()


def test_error_paths(pkg, cfg0):
    tf = cfg0
    P = tf.params
    # row out of range -> TPCCA_E_RANGE at sync
    trk = pkg.Tracker(P, max_clusters=16)
    trk.load_clusters(0, np.zeros(3, np.float32), np.ones(3, np.float32), np.array([1, 2, 999], np.uint16))
    trk.run()
    with pytest.raises(pkg.TpccaError) as e:
        trk.sync()
    assert e.value.code == -5
    trk.close()
    # the same with a workspace full of 0x7f bytes and good clusters around the bad one: the positions S1 / S2 never
    # wrote hold garbage "links"; S3-S5 must not follow them (illegal-address fault instead of E_RANGE)
    row = tf.row[0].copy(); row[len(row) // 2] = 400
    for fill in (0x7f, 0xff, 0x00):
        trk = pkg.Tracker(P, max_clusters=tf.n_clusters, workspace_fill=fill)
        trk.load_clusters(0, tf.y[0], tf.z[0], row)
        trk.run()
        with pytest.raises(pkg.TpccaError) as e:
            trk.sync()
        assert e.value.code == -5
        # the context (and the CUDA context of the process) is still usable
        trk.load_timeframe(tf)
        trk.run()
        compare_timeframe(trk, tf, Oracle(P))
        trk.close()
    trk = pkg.Tracker(P, max_clusters=16)
    # loading a sector twice -> E_STATE; too many clusters -> E_WORKSPACE
    trk.reset()
    trk.load_clusters(0, np.zeros(3, np.float32), np.ones(3, np.float32), np.array([1, 2, 3], np.uint16))
    with pytest.raises(pkg.TpccaError) as e:
        trk.load_clusters(0, np.zeros(3, np.float32), np.ones(3, np.float32), np.array([1, 2, 3], np.uint16))
    assert e.value.code == -2
    trk.reset()
    with pytest.raises(pkg.TpccaError) as e:
        trk.load_clusters(0, np.zeros(30, np.float32), np.ones(30, np.float32), np.zeros(30, np.uint16))
    assert e.value.code == -4
    # S2 before S1 -> E_STATE
    trk.reset()
    trk.load_clusters(0, np.zeros(3, np.float32), np.ones(3, np.float32), np.array([1, 2, 3], np.uint16))
    with pytest.raises(pkg.TpccaError) as e:
        trk.run(2)
    assert e.value.code == -2
    trk.close()
    # start-hit capacity overflow is reported, never silently truncated
    trk = pkg.Tracker(P, max_clusters=tf.n_clusters, max_start_hits=5)
    trk.load_timeframe(tf)
    trk.run()
    with pytest.raises(pkg.TpccaError) as e:
        trk.sync()
    assert e.value.code == -4
    trk.close()


def test_device_inputs_and_borrow(pkg, cfg0):
    """Clusters already resident in HBM (torch CUDA tensors): copy and borrow modes."""
    import torch
    tf = cfg0
    y = torch.from_numpy(tf.y[0]).cuda(); z = torch.from_numpy(tf.z[0]).cuda()
    row = torch.from_numpy(tf.row[0].astype(np.int16)).cuda().view(torch.uint16)
    orc = Oracle(tf.params)
    for borrow in (False, True):
        trk = pkg.Tracker(tf.params, max_clusters=tf.n_clusters)
        trk.load_clusters(0, y, z, row, borrow=borrow)
        trk.run()
        compare_timeframe(trk, tf, orc)
        trk.close()


def test_early_fetch_while_s5_runs(pkg, cfg1_small):
    """HOST fetch of the S1-S4 outputs right after tpcca_run (it waits for S4 only and overlaps S5) delivers
    the same arrays as the fetch after the whole run."""
    from paper_2208_07412_b200 import binding as B
    tf = cfg1_small
    trk = pkg.Tracker(tf.params, max_clusters=tf.n_clusters)
    trk.load_timeframe(tf)
    trk.run()
    early = [trk.get_tracks(s, B.OUT_ORDER | B.OUT_LINKS | B.OUT_START) for s in (0, 7, 35)]
    full = [trk.get_tracks(s) for s in (0, 7, 35)]
    for a, b in zip(early, full):
        assert a.x_ref is None and a.n_tracks == 0 and b.n_tracks > 0
        for f in ("order", "link_up", "link_dn", "start_hit"):
            assert np.array_equal(getattr(a, f), getattr(b, f)), f
    compare_timeframe(trk, tf, Oracle(tf.params), sectors=(0, 7, 35))
    trk.close()


def test_config1_full_size(pkg):
    """BASELINE.json config 1 at full size (10k tracks, ~1.5M clusters): every sector, every output."""
    tf = tpcsynth.generate(1)
    assert tf.n_clusters > 1_000_000
    rep = check(pkg, tf)
    assert rep["n_tracks"] > 20000 and rep["links_differing"] == 0


# ------------------------------------------------------------------------------------------------
# kernel instances / capacities / sizes the small cases above never select
# ------------------------------------------------------------------------------------------------
def test_large_capacity_selects_dense_instances(pkg, cfg0):
    """A context whose CAPACITY exceeds 0.7 clusters per grid bin takes the S2 variant for dense time frames
    and, above ~700 clusters per coarse bucket, the smallest S1 slab (slab_shift 5): both must give the oracle's
    outputs.  Asserted through tpcca_get_info."""
    tf = cfg0
    small = pkg.Tracker(tf.params, max_clusters=tf.n_clusters)
    big = pkg.Tracker(tf.params, max_clusters=120_000)
    a, b = small.info(), big.info()
    small.close()
    assert b["slab_shift"] == 5 and a["slab_shift"] > 5
    assert b["s2_variant"] > a["s2_variant"]
    big.load_timeframe(tf)
    big.run()
    rep = compare_timeframe(big, tf, Oracle(tf.params))
    big.close()
    assert rep["n_tracks"] > 100 and rep["links_differing"] == 0


def test_dense_uniform_sector(pkg):
    """A genuinely dense input: 72k uniform clusters on 12 rows of one sector (about 1.3 clusters per bin on those
    rows; S2 windows with tens of candidates, hit lists overflowing, S5 searches over long candidate lists), in a
    context sized for it (dense S2 variant)."""
    P = tpcsynth.default_params(n_sectors=1)
    rng = np.random.default_rng(17)
    n = 72_000
    row = rng.integers(20, 32, n).astype(np.uint16)
    y = ((rng.random(n) * 2.0 - 1.0) * 17.0).astype(np.float32)
    z = (rng.random(n) * 250.0).astype(np.float32)
    tf = ArrTF(P, [(y, z, row)])
    trk = run_gpu(pkg, tf, max_start_hits=n // 2)
    assert trk.info()["s2_variant"] >= 15
    rep = compare_timeframe(trk, tf, Oracle(P))
    trk.close()
    assert rep["links_differing"] == 0


def test_full_time_frame_axis_128_orbits(pkg):
    """The 29 617 cm z axis of BASELINE.json configs[3] with its full grid tables (10.3 M bins per sector):
    collisions at t = 0, T/2 and T (fp32 ulp of z is 2e-3 cm at the far end: K-rule Z and the bin keys are the
    parts that depend on it).  All 36 sectors, every output."""
    T = 128 * tpcsynth.ORBIT_US
    tf = tpcsynth.generate(3, coll_times=[0.0, 0.013, 0.5 * T, 0.5 * T + 31.0, T - 0.02, T], coll_mult=700)
    assert max(float(z.max()) for z in tf.z) > 29_500.0 and tf.params.bins_per_sector() > 10_000_000
    rep = check(pkg, tf)
    assert rep["sectors"] == 36 and rep["n_tracks"] > 4000 and rep["links_differing"] == 0


def test_config4_full_size(pkg):
    """BASELINE.json configs[4] at full size (15k tracks, ~2.1 M clusters, 20 % noise, loopers): all sectors."""
    tf = tpcsynth.generate(4)
    assert tf.n_clusters > 1_800_000
    rep = check(pkg, tf)
    assert rep["sectors"] == 36 and rep["n_tracks"] > 20000 and rep["links_differing"] == 0


def test_config2_full_size_six_sectors(pkg):
    """BASELINE.json configs[2] at full size (32 orbits, ~3.6e7 clusters) on the GPU; six sectors spread over
    both sides are compared element by element with the oracle."""
    tf = tpcsynth.generate(2)
    assert tf.n_clusters > 25_000_000
    rep = check(pkg, tf, sectors=(0, 7, 13, 18, 26, 35))
    assert rep["sectors"] == 6 and rep["n_clusters"] > 4_000_000 and rep["links_differing"] == 0


# ------------------------------------------------------------------------------------------------
# S6 tracklet selector
# ------------------------------------------------------------------------------------------------
def run_gpu_select(pkg, tf, **kw):
    trk = pkg.Tracker(tf.params, max_clusters=max(tf.n_clusters, 1), workspace_fill=WS_FILL, **kw)
    trk.load_timeframe(tf)
    trk.run(0x3F)
    trk.sync()
    return trk


def test_selector_config0_and_config1(pkg, cfg0, cfg1_small):
    from parity import compare_selection
    for tf in (cfg0, cfg1_small):
        trk = run_gpu_select(pkg, tf)
        orc = Oracle(tf.params)
        compare_timeframe(trk, tf, orc)                    # S1-S5 outputs are untouched by S6
        rep = compare_selection(trk, tf, orc)
        cnt = trk.counts()
        assert cnt["n_selected"] == rep["n_selected"] and 0 < rep["n_selected"] < rep["n_tracks"]
        assert trk.timings()[6] > 0.0
        trk.close()


def test_selector_separate_run_and_thresholds(pkg, cfg1_small):
    """S6 on its own after an S1-S5 run; other thresholds (0 = no shared hit allowed, 1000 = keep all)."""
    from parity import compare_selection
    tf = cfg1_small
    for permille in (0, 250, 1000):
        P = tf.params.copy(sel_max_shared_permille=permille)
        tf2 = ArrTF(P, [(tf.y[s], tf.z[s], tf.row[s]) for s in (2, 11, 29)])
        trk = run_gpu(pkg, tf2)
        trk.run(0x20)
        trk.sync()
        rep = compare_selection(trk, tf2, Oracle(P))
        if permille == 1000:
            assert rep["n_selected"] == rep["n_tracks"]
        # re-running S5 alone invalidates the selection (its tables alias S5 scratch)
        trk.run(0x10)
        trk.sync()
        assert trk.counts()["n_selected"] == 0
        trk.close()


def test_selector_dense_stress_and_empty(pkg):
    from parity import compare_selection
    tf = tpcsynth.generate(4, n_tracks=1500)
    trk = run_gpu_select(pkg, tf)
    rep = compare_selection(trk, tf, Oracle(tf.params))
    assert rep["n_selected"] > 300
    trk.close()
    P = tpcsynth.default_params(n_sectors=3)
    e = (np.empty(0, np.float32), np.empty(0, np.float32), np.empty(0, np.uint16))
    one = (np.array([0.5], np.float32), np.array([10.0], np.float32), np.array([7], np.uint16))
    for secs in ([e, e, e], [one, e, one]):
        tf = ArrTF(P, secs)
        trk = run_gpu_select(pkg, tf)
        assert compare_selection(trk, tf, Oracle(P))["n_selected"] == 0
        trk.close()
    rng = np.random.default_rng(2)
    n = 6000
    tf = ArrTF(tpcsynth.default_params(n_sectors=1), [((rng.random(n) * 16.0 - 8.0).astype(np.float32),
                                                       (rng.random(n) * 12.0).astype(np.float32),
                                                       rng.integers(0, 12, n).astype(np.uint16))])
    trk = run_gpu_select(pkg, tf)
    compare_selection(trk, tf, Oracle(tf.params))
    trk.close()


# ------------------------------------------------------------------------------------------------
# S7 track-residual front end
# ------------------------------------------------------------------------------------------------
def test_residuals_config0_config1_config4(pkg, cfg0, cfg1_small):
    from parity import compare_residuals, compare_selection
    for tf in (cfg0, cfg1_small, tpcsynth.generate(4, n_tracks=1500)):
        trk = pkg.Tracker(tf.params, max_clusters=tf.n_clusters)
        trk.load_timeframe(tf)
        trk.run(0x7F)
        trk.sync()
        orc = Oracle(tf.params)
        rep = compare_residuals(trk, tf, orc)
        assert rep["n_attached"] > 0.7 * rep["n_clusters"]
        compare_selection(trk, tf, orc)
        assert trk.timings()[7] > 0.0
        trk.close()


def test_residuals_separate_run_quantum_and_empty(pkg, cfg1_small):
    from parity import compare_residuals
    tf = cfg1_small
    P = tf.params.copy(res_inv_quantum=32.0, sel_max_shared_permille=300)
    tf2 = ArrTF(P, [(tf.y[s], tf.z[s], tf.row[s]) for s in (4, 22)])
    trk = run_gpu(pkg, tf2)
    trk.run(0x20)
    trk.run(0x40)
    trk.sync()
    compare_residuals(trk, tf2, Oracle(P))
    trk.close()
    P3 = tpcsynth.default_params(n_sectors=2)
    e = (np.empty(0, np.float32), np.empty(0, np.float32), np.empty(0, np.uint16))
    one = (np.array([0.5], np.float32), np.array([10.0], np.float32), np.array([7], np.uint16))
    tf3 = ArrTF(P3, [e, one])
    trk = pkg.Tracker(P3, max_clusters=4)
    trk.load_timeframe(tf3)
    trk.run(0x7F)
    trk.sync()
    compare_residuals(trk, tf3, Oracle(P3))
    trk.close()


# ------------------------------------------------------------------------------------------------
# time-frame streaming: sector-group pipeline
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_groups", [1, 4, 5])
def test_pipeline_equals_oracle(pkg, cfg1_small, n_groups):
    """Every sector delivered by the pipeline (S1-S7 per sector group on its own stream / thread) equals the
    oracle element by element; 5 groups: uneven group sizes (36 sectors)."""
    from paper_2208_07412_b200 import binding as B
    from parity import _eq
    tf = cfg1_small
    cap = int(max(tf.sector_counts().reshape(-1).sum() // n_groups * 1.5, 1000))
    pipe = pkg.Pipeline(tf.params, n_groups, max_clusters_group=cap)
    first, _ = pipe.groups()
    assert first[0] == 0 and first[-1] == 36 and len(first) == n_groups + 1
    what = B.OUT_ALL | B.OUT_SELECTION | B.OUT_RESIDUALS
    orc = Oracle(tf.params)
    for rep in range(2):                       # a pipeline is reusable: second time frame through the same contexts
        outs = pipe.run(tf.y, tf.z, tf.row, stage_mask=0x7F, what=what)
        for s in (range(36) if rep == 0 else (0, 17, 35)):
            o = orc.run(tf.y[s], tf.z[s], tf.row[s], stage_mask=0x7F)
            try:
                compare_sector(outs[s], o, orc, tf.row[s][o.order])
                r = {}
                _eq("owner", outs[s].owner, o.owner, r); _eq("selected", outs[s].selected, o.selected, r)
                _eq("res_trk", outs[s].res_trk, o.res_trk, r); _eq("q_y", outs[s].q_y, o.q_y, r)
            except ParityError as e:
                raise ParityError(f"groups {n_groups} sector {s}: {e}") from None
    pipe.close()


def test_pipeline_device_inputs_and_errors(pkg, cfg1_small):
    import torch
    from paper_2208_07412_b200 import binding as B
    tf = cfg1_small
    pipe = pkg.Pipeline(tf.params, 3, max_clusters_group=tf.n_clusters)
    y = [torch.from_numpy(a).cuda() for a in tf.y]; z = [torch.from_numpy(a).cuda() for a in tf.z]
    row = [torch.from_numpy(a.astype(np.int16)).cuda().view(torch.uint16) for a in tf.row]
    outs = pipe.run(y, z, row)
    orc = Oracle(tf.params)
    for s in (5, 20):
        o = orc.run(tf.y[s], tf.z[s], tf.row[s])
        compare_sector(outs[s], o, orc, tf.row[s][o.order])
    pipe.close()
    # a group whose capacity is too small reports it (nothing is truncated)
    pipe = pkg.Pipeline(tf.params, 4, max_clusters_group=1000)
    with pytest.raises(pkg.TpccaError) as e:
        pipe.run(tf.y, tf.z, tf.row)
    assert e.value.code == -4 and "group" in str(e.value)
    pipe.close()
    with pytest.raises(pkg.TpccaError):
        pkg.Pipeline(tf.params, 99, max_clusters_group=1000)


def test_pipeline_device_inputs_still_being_written(pkg, cfg1_small):
    """Device inputs whose upload is still queued on the caller's stream when the pipeline is called: the groups'
    streams must wait for it (they used to copy at once and could read the buffers before the data had arrived)."""
    import torch
    tf = cfg1_small
    pipe = pkg.Pipeline(tf.params, 3, max_clusters_group=tf.n_clusters)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hy = [pin(a) for a in tf.y]; hz = [pin(a) for a in tf.z]; hr = [pin(a.astype(np.int16)) for a in tf.row]
    y = [torch.zeros_like(a, device="cuda") for a in hy]; z = [torch.zeros_like(a, device="cuda") for a in hz]
    row = [torch.zeros_like(a, device="cuda") for a in hr]
    torch.cuda.synchronize()
    torch.cuda._sleep(400_000_000)                  # ~0.2 s of busy waiting on the current stream, then the uploads
    for d, h in zip(y + z + row, hy + hz + hr):
        d.copy_(h, non_blocking=True)
    outs = pipe.run(y, z, [r.view(torch.uint16) for r in row])
    orc = Oracle(tf.params)
    for s in (0, 13, 35):
        o = orc.run(tf.y[s], tf.z[s], tf.row[s])
        compare_sector(outs[s], o, orc, tf.row[s][o.order])
    pipe.close()


def test_pipeline_refuses_merge_and_shared_streams(pkg, cfg1_small):
    """S8 crosses sectors and a group only knows its own: the pipeline refuses it (it used to run it per group, with
    links over group boundaries missing and group-local sector numbers).  Any two groups on one stream are refused at
    create, not only neighbouring ones."""
    import ctypes as C
    import torch
    from paper_2208_07412_b200 import binding as B
    tf = cfg1_small
    pipe = pkg.Pipeline(tf.params, 2, max_clusters_group=tf.n_clusters)       # 2 x 18 sectors: group = TPC side
    for mask, what in ((0xFF, B.OUT_ALL), (0x7F, B.OUT_ALL | B.OUT_MERGE), (0xFF, B.OUT_ALL | B.OUT_MERGE)):
        with pytest.raises(pkg.TpccaError) as e:
            pipe.run(tf.y, tf.z, tf.row, stage_mask=mask, what=what)
        assert e.value.code == -1 and "MERGE" in str(e.value)
    outs = pipe.run(tf.y, tf.z, tf.row, stage_mask=0x7F, what=B.OUT_ALL | B.OUT_SELECTION)   # still usable afterwards
    assert sum(o.n_tracks for o in outs) > 1000 and all(o.merge is None for o in outs)
    lib = pkg.load_library()
    p, keep = B._make_params(tf.params)
    a, b = torch.cuda.Stream(), torch.cuda.Stream()
    nbytes = pipe.workspace_bytes_each                                         # sized for 18 sectors: enough for 12
    ws = [torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda:0") for _ in range(3)]
    wsp = (C.c_void_p * 3)(*[(w.data_ptr() + 255) // 256 * 256 for w in ws])
    for order, ok in (((a, b, a), False), ((a, a, b), False), ((a, b, torch.cuda.Stream()), True)):
        st = (C.c_void_p * 3)(*[x.cuda_stream for x in order])
        h = C.c_void_p()
        rc = lib.tpcca_pipeline_create(C.byref(p), 0, 3, st, wsp, nbytes, tf.n_clusters, 0, C.byref(h))
        if ok:
            assert rc == 0 and h.value
            lib.tpcca_pipeline_destroy(h)
        else:
            assert rc == -1 and not h.value and "own stream" in lib.tpcca_pipeline_last_error(None).decode()
    pipe.close()


def test_timings_are_zero_for_stages_not_run(pkg, cfg1_small):
    """tpcca_get_timings: a stage outside the run's mask reports exactly 0 (the events around it are recorded all the
    same, microseconds apart)."""
    tf = cfg1_small
    trk = pkg.Tracker(tf.params, max_clusters=tf.n_clusters)
    trk.load_timeframe(tf)
    trk.run(0x03); trk.sync()
    t = trk.timings()
    assert t[0] > 0 and t[1] > 0 and t[5] > 0 and t[2] == t[3] == t[4] == t[6] == t[7] == t[8] == 0.0
    trk.run(0x1C); trk.sync()                       # S3-S5 on top of the S1 / S2 outputs
    t = trk.timings()
    assert t[0] == t[1] == 0.0 and min(t[2:6]) > 0 and t[6] == t[7] == t[8] == 0.0
    trk.run(0x7F); trk.sync()
    t = trk.timings()
    assert min(t[:8]) > 0 and t[8] == 0.0           # S8 not run: 0, not the gap between two event records
    t1 = trk.timings(2)
    assert t1[0] > 0 and t1[2] == 0.0               # the ring keeps each run's own mask
    trk.close()


def test_get_tracks_all_equals_per_sector(pkg, cfg1_small):
    tf = cfg1_small
    trk = run_gpu(pkg, tf)
    allv = trk.get_tracks_all()
    for s in (0, 9, 35):
        one = trk.get_tracks(s)
        for f in ("order", "link_up", "start_hit", "par", "cov", "hit_idx", "hit_offset"):
            assert np.array_equal(getattr(allv[s], f), getattr(one, f)), f
    trk.close()


# ------------------------------------------------------------------------------------------------
# S8 cross-sector merging + chain refit
# ------------------------------------------------------------------------------------------------
def test_merge_config1_and_config4(pkg, cfg1_small):
    from parity import compare_merge
    for tf in (cfg1_small, tpcsynth.generate(1, n_tracks=4000), tpcsynth.generate(4, n_tracks=2500)):
        trk = pkg.Tracker(tf.params, max_clusters=tf.n_clusters, workspace_fill=WS_FILL)
        trk.load_timeframe(tf)
        trk.run(0xFF)
        trk.sync()
        rep = compare_merge(trk, tf)
        assert rep["n_links"] > 0.2 * rep["n_selected"] and rep["n_chains"] > 0
        t = trk.timings()
        assert all(v > 0.0 for v in t)           # every stage of mask 0xFF ran and was timed
        compare_timeframe(trk, tf, Oracle(tf.params), sectors=(0, 19))       # S1-S5 outputs untouched by S6-S8
        trk.close()


def _mirror_track(rows, y0, sign, z0=100.0):
    """Clusters of one straight-ish track on rows [rows[0], rows[1]): y = sign * (y0 + eps_row) with dyadic eps, z = z0.
    sign = -1 is the exact y mirror image (negation is exact in every operation of the filter); y0 = 0: y == 0."""
    rows = np.arange(*rows)
    eps = ((rows * 7) % 5 - 2) / 64.0 if y0 else 0.0
    return rows.astype(np.uint16), (sign * (y0 + eps) * np.ones(len(rows))).astype(np.float32), np.full(len(rows), z0, np.float32)


def test_merge_ties_through_real_clusters(pkg):
    """The S8 tie-breaks of the CUDA path (the 64-bit atomicMin key order of k_mg_match), through real clusters.
    Three sectors of one side with the identity as sector rotation: a track at y == 0 has two partner candidates that
    are exact y-mirror images of each other (+-2 cm), so dy and ds tie bit for bit and the score ties; the definition
    picks the smaller sector, then the smaller track.  Ties for next() (two upper candidates) and for
    prev() (two lower candidates), within one neighbour sector and across the two neighbour sectors (either way round:
    the kernel visits sector 2 before sector 0)."""
    from oracle import run_timeframe_merged
    from parity import compare_merge
    P = tpcsynth.default_params(n_sectors=3).copy(sectors_per_side=3, sector_cos=1.0, sector_sin=0.0, mg_dy=4.0)
    LO, UP = (5, 41), (43, 80)
    #        centre track     first candidate   its mirror image    expected partner (sector, track)
    cases = [((1, LO, 0.0, 1), (2, UP, 2.0, 1), (2, UP, 2.0, -1), "next", (2, 0)),
             ((1, LO, 0.0, 1), (2, UP, 2.0, 1), (0, UP, 2.0, -1), "next", (0, 0)),
             ((1, LO, 0.0, 1), (0, UP, 2.0, 1), (2, UP, 2.0, -1), "next", (0, 0)),
             ((1, UP, 0.0, 1), (0, LO, 2.0, 1), (0, LO, 2.0, -1), "prev", (0, 0)),
             ((1, UP, 0.0, 1), (0, LO, 2.0, 1), (2, LO, 2.0, -1), "prev", (0, 0)),
             ((1, UP, 0.0, 1), (2, LO, 2.0, 1), (0, LO, 2.0, -1), "prev", (0, 0))]
    for *placement, which, want in cases:
        secs = [([], [], []) for _ in range(3)]
        for sec, rows, y0, sign in placement:
            r, y, z = _mirror_track(rows, y0, sign)
            secs[sec][0].append(y); secs[sec][1].append(z); secs[sec][2].append(r)
        cat = lambda l, dt: np.concatenate(l).astype(dt) if l else np.zeros(0, dt)
        tf = ArrTF(P, [(cat(a, np.float32), cat(b, np.float32), cat(c, np.uint16)) for a, b, c in secs])
        # the premise, on the oracle: the two candidates are fitted to exact mirror images, and the tie goes to `want`
        res, mg = run_timeframe_merged(tf, "f32")
        cand = [res[sec].par[res[sec].selected] for sec, *_ in placement[1:]]
        both = np.concatenate(cand) if placement[1][0] != placement[2][0] else cand[0]
        assert both.shape == (2, 5) and np.array_equal(both[0] * [-1, 1, -1, 1, -1], both[1]) and both[0, 0] != 0.0
        m1 = mg[1]
        got = (int(m1.next_sec[0]), int(m1.next_trk[0])) if which == "next" else (int(m1.prev_sec[0]), int(m1.prev_trk[0]))
        assert got == want, (placement, got, want)
        # the CUDA path makes the same choice (links bit-exact, chains and refits compared as everywhere)
        trk = pkg.Tracker(P, max_clusters=tf.n_clusters, workspace_fill=WS_FILL)
        trk.load_timeframe(tf)
        trk.run(0xFF)
        trk.sync()
        rep = compare_merge(trk, tf)
        assert rep["n_links"] == 1 and rep["n_chains"] == 1, rep
        trk.close()


def test_merge_full_occupancy_three_sectors(pkg):
    """S8 against the oracle at the FULL occupancy of the time-frame configs (the bench checks S8 at full size by
    properties only: the oracle's all-pairs matching is out of reach over 36 sectors x 128 orbits).  Three neighbouring
    sectors of BASELINE.json configs[2] at full size (32 orbits at 50 kHz: the same clusters per cm of drift as
    configs[3]), ~1.35 M clusters and ~19 k selected tracks each, as a three-sector side: ~2e9 pair tests in the oracle.
    Links bit-exact, chains walked along the tracker's links, refits within 1e-4."""
    from parity import compare_merge
    full = tpcsynth.generate(2)
    P = full.params.copy(n_sectors=3, sectors_per_side=3)
    tf = ArrTF(P, [(full.y[s], full.z[s], full.row[s]) for s in (0, 1, 2)])
    assert tf.n_clusters > 3_000_000
    trk = pkg.Tracker(P, max_clusters=tf.n_clusters, workspace_fill=WS_FILL)
    trk.load_timeframe(tf)
    trk.run(0xFF)
    trk.sync()
    rep = compare_merge(trk, tf)
    assert rep["n_selected"] > 50_000 and rep["n_links"] > 15_000 and rep["n_chains"] > 12_000, rep
    trk.close()


def test_merge_time_frame_and_degenerate_layouts(pkg):
    """Several collisions along the 128-orbit z axis (candidate index over 900+ z buckets); sector layouts without a
    neighbour relation (1 or 3 sectors: S8 is a no-op) and with two sectors per side."""
    from parity import compare_merge
    T = 128 * tpcsynth.ORBIT_US
    tf = tpcsynth.generate(3, coll_times=[0.0, 0.2 * T, 0.2 * T + 9.0, 0.77 * T, T], coll_mult=900)
    trk = pkg.Tracker(tf.params, max_clusters=tf.n_clusters)
    trk.load_timeframe(tf)
    trk.run(0xFF)
    trk.sync()
    rep = compare_merge(trk, tf)
    assert rep["n_links"] > 500
    trk.close()
    base = tpcsynth.generate(1, n_tracks=1500)
    for nsec, per in ((1, 18), (3, 18), (4, 2), (6, 3)):
        P = base.params.copy(n_sectors=nsec, sectors_per_side=per)
        tf2 = ArrTF(P, [(base.y[s], base.z[s], base.row[s]) for s in range(nsec)])
        trk = pkg.Tracker(P, max_clusters=tf2.n_clusters)
        trk.load_timeframe(tf2)
        trk.run(0xFF)
        trk.sync()
        rep = compare_merge(trk, tf2)
        if nsec % per:
            assert rep["n_links"] == 0
        trk.close()


def test_dense_slice_all_stages(pkg):
    """S6-S8 at the occupancy of the ~4e8-cluster footprint (one orbit of the time-frame recipe at 2.75x
    multiplicity, 36 sectors): selection, residual codes and merge links bit-exact, chain refits within 1e-4."""
    from parity import compare_merge, compare_residuals, compare_selection
    tf = tpcsynth.generate(2, n_orbits=1, mult_scale=2.75, seed=220807499)
    trk = pkg.Tracker(tf.params, max_clusters=tf.n_clusters, workspace_fill=WS_FILL)
    trk.load_timeframe(tf)
    trk.run(0xFF)
    trk.sync()
    orc = Oracle(tf.params)
    sel = compare_selection(trk, tf, orc, sectors=(0, 8, 17, 18, 30))
    assert sel["n_selected"] > 200
    compare_residuals(trk, tf, orc, sectors=(3, 21))
    rep = compare_merge(trk, tf)
    assert rep["n_links"] > 300 and rep["n_chains"] > 200
    trk.close()
