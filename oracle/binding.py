"""ctypes binding of liboracle.so (TEST INFRASTRUCTURE; see tpcca_oracle.cpp header)."""
from __future__ import annotations

import ctypes as C
import dataclasses

import numpy as np

from . import build as _build

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class _Params(C.Structure):
    _fields_ = [
        ("n_rows", C.c_int32),
        ("row_x", _dp), ("grid_y_lo", _dp), ("grid_inv_bin_y", _dp), ("grid_ny", _ip),
        ("grid_z_lo", C.c_double), ("grid_inv_bin_z", _dp), ("grid_nz", _ip),
        ("nf_hy_up", _dp), ("nf_hz_up", _dp), ("nf_hy_dn", _dp), ("nf_hz_dn", _dp), ("nf_cut", _dp),
        ("kappa_per_qpt", C.c_double), ("err2_y", C.c_double), ("err2_z", C.c_double),
        ("init_cov", C.c_double * 5),
        ("tc_win_y", C.c_double), ("tc_win_z", C.c_double), ("tc_gate", C.c_double),
        ("max_sinphi", C.c_double), ("grid_margin", C.c_double),
        ("tc_max_gap", C.c_int32), ("tc_min_hits", C.c_int32),
        ("sel_max_shared_permille", C.c_int32), ("res_inv_quantum", C.c_double),
        ("sectors_per_side", C.c_int32), ("sector_cos", C.c_double), ("sector_sin", C.c_double),
        ("mg_max_row_gap", C.c_int32), ("mg_dy", C.c_double), ("mg_dz", C.c_double), ("mg_dsin", C.c_double),
        ("mg_zpre", C.c_double),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        lib.oracle_create.restype = C.c_void_p
        lib.oracle_create.argtypes = [C.POINTER(_Params), C.c_int]
        lib.oracle_destroy.argtypes = [C.c_void_p]
        lib.oracle_load.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.oracle_run.argtypes = [C.c_void_p, C.c_uint32, C.c_int]
        lib.oracle_sizes.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
        lib.oracle_get_grid.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        lib.oracle_get_links.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        lib.oracle_get_tracks.argtypes = [C.c_void_p] + [C.c_void_p] * 8
        lib.oracle_kf_propagate.argtypes = [C.c_void_p, _dp, C.c_double]
        lib.oracle_kf_propagate.restype = C.c_int
        lib.oracle_kf_update.argtypes = [C.c_void_p, _dp, C.c_double, C.c_double]
        lib.oracle_kf_dist2.argtypes = [C.c_void_p, _dp, C.c_double, C.c_double]
        lib.oracle_kf_dist2.restype = C.c_double
        lib.oracle_score.argtypes = [C.c_void_p, C.c_int] + [C.c_double] * 6
        lib.oracle_score.restype = C.c_double
        lib.oracle_n_selected.argtypes = [C.c_void_p]
        lib.oracle_n_selected.restype = C.c_int64
        lib.oracle_get_selection.argtypes = [C.c_void_p] + [C.c_void_p] * 3
        lib.oracle_merge.argtypes = [C.POINTER(C.c_void_p), C.c_int]
        lib.oracle_inject_selected.argtypes = [C.c_void_p, C.c_int32] + [C.c_void_p] * 4
        lib.oracle_get_merge_links.argtypes = [C.c_void_p] + [C.c_void_p] * 4 + [C.POINTER(C.c_int64)]
        lib.oracle_get_merged.argtypes = [C.c_void_p] + [C.c_void_p] * 9
        lib.oracle_kf_rotate.argtypes = [C.c_void_p, _dp, C.c_double, C.c_double]
        lib.oracle_kf_rotate.restype = C.c_int
        lib.oracle_get_residuals.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        lib.oracle_select.argtypes = [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_int32] + [C.c_void_p] * 3
        lib.oracle_select.restype = C.c_int64
        _lib = lib
    return _lib


@dataclasses.dataclass
class OracleResult:
    """Outputs of one sector.  Index space: sorted positions (after S1); order: sorted -> original."""
    n: int
    order: np.ndarray = None
    sy: np.ndarray = None
    sz: np.ndarray = None
    bin_start: np.ndarray = None
    row_start: np.ndarray = None
    link_up_raw: np.ndarray = None
    link_dn_raw: np.ndarray = None
    link_up: np.ndarray = None
    link_dn: np.ndarray = None
    start_hit: np.ndarray = None
    x_ref: np.ndarray = None
    z_ref: np.ndarray = None
    par: np.ndarray = None       # [n_tracks, 5]
    cov: np.ndarray = None       # [n_tracks, 15]
    chi2: np.ndarray = None
    n_hits: np.ndarray = None
    n_fit: np.ndarray = None
    first_row: np.ndarray = None
    last_row: np.ndarray = None
    trk_start_hit: np.ndarray = None
    hit_offset: np.ndarray = None
    hit_idx: np.ndarray = None
    owner: np.ndarray = None        # S6: [n] track owning each cluster (-1 none)
    n_own: np.ndarray = None        # S6: [n_tracks]
    selected: np.ndarray = None     # S6: [n_selected] ascending track numbers
    res_trk: np.ndarray = None      # S7: [n] selected track owning the cluster (-1: stored raw)
    res_y: np.ndarray = None        # S7: [n] residuals to the track model
    res_z: np.ndarray = None
    q_y: np.ndarray = None          # S7: [n] int16 quantised residuals
    q_z: np.ndarray = None

    @property
    def n_tracks(self) -> int:
        return 0 if self.x_ref is None else int(self.x_ref.shape[0])


def _d(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


class Oracle:
    """One oracle instance = one set of tables; `run` processes one sector."""

    def __init__(self, params, precision: str = "f32"):
        lib = _load()
        self._lib = lib
        self.precision = {"f32": 0, "f64": 1}[precision]
        self.n_rows = int(params.n_rows)
        self._keep = dict(
            row_x=_d(params.row_x), grid_y_lo=_d(params.grid_y_lo),
            grid_inv_bin_y=_d(params.grid_inv_bin_y), grid_inv_bin_z=_d(params.grid_inv_bin_z),
            nf_hy_up=_d(params.nf_hy_up), nf_hz_up=_d(params.nf_hz_up),
            nf_hy_dn=_d(params.nf_hy_dn), nf_hz_dn=_d(params.nf_hz_dn), nf_cut=_d(params.nf_cut),
            grid_ny=np.ascontiguousarray(params.grid_ny, dtype=np.int32),
            grid_nz=np.ascontiguousarray(params.grid_nz, dtype=np.int32))
        k = self._keep
        p = _Params()
        p.n_rows = self.n_rows
        for name in ("row_x", "grid_y_lo", "grid_inv_bin_y", "grid_inv_bin_z", "nf_hy_up", "nf_hz_up",
                     "nf_hy_dn", "nf_hz_dn", "nf_cut"):
            setattr(p, name, k[name].ctypes.data_as(_dp))
        p.grid_ny = k["grid_ny"].ctypes.data_as(_ip)
        p.grid_nz = k["grid_nz"].ctypes.data_as(_ip)
        p.grid_z_lo = float(params.grid_z_lo)
        p.kappa_per_qpt = float(params.kappa_per_qpt)
        p.err2_y = float(params.err2_y)
        p.err2_z = float(params.err2_z)
        for i in range(5):
            p.init_cov[i] = float(params.init_cov[i])
        p.tc_win_y = float(params.tc_win_y); p.tc_win_z = float(params.tc_win_z)
        p.tc_gate = float(params.tc_gate); p.max_sinphi = float(params.max_sinphi)
        p.grid_margin = float(params.grid_margin)
        p.tc_max_gap = int(params.tc_max_gap); p.tc_min_hits = int(params.tc_min_hits)
        p.sel_max_shared_permille = int(getattr(params, "sel_max_shared_permille", 500))
        p.res_inv_quantum = float(getattr(params, "res_inv_quantum", 128.0))
        p.sectors_per_side = int(getattr(params, "sectors_per_side", 18))
        p.sector_cos = float(getattr(params, "sector_cos", np.float32(np.cos(np.pi / 9))))
        p.sector_sin = float(getattr(params, "sector_sin", np.float32(np.sin(np.pi / 9))))
        p.mg_max_row_gap = int(getattr(params, "mg_max_row_gap", 8))
        p.mg_dy = float(getattr(params, "mg_dy", 1.0)); p.mg_dz = float(getattr(params, "mg_dz", 1.0))
        p.mg_dsin = float(getattr(params, "mg_dsin", 0.05)); p.mg_zpre = float(getattr(params, "mg_zpre", 32.0))
        self._h = lib.oracle_create(C.byref(p), self.precision)
        if not self._h:
            raise RuntimeError("oracle_create failed")

    def close(self):
        if getattr(self, "_h", None):
            self._lib.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    # ------------------------------------------------------------------------------
    def run(self, y, z, row, stage_mask: int = 0x1F, brute: bool = False, want=("grid", "links", "tracks")) -> OracleResult:
        ft = np.float32 if self.precision == 0 else np.float64
        y = np.ascontiguousarray(y, dtype=ft)
        z = np.ascontiguousarray(z, dtype=ft)
        row = np.ascontiguousarray(row, dtype=np.uint16)
        n = int(y.shape[0])
        rc = self._lib.oracle_load(self._h, n, y.ctypes.data, z.ctypes.data, row.ctypes.data)
        if rc != 0:
            raise ValueError(f"oracle_load failed: {rc}")
        self._lib.oracle_run(self._h, stage_mask, int(brute))
        sizes = (C.c_int64 * 5)()
        self._lib.oracle_sizes(self._h, sizes)
        _, n_start, n_trk, n_hit, n_bins = (int(v) for v in sizes)
        res = OracleResult(n=n)
        if "grid" in want and (stage_mask & 1):
            res.order = np.empty(n, np.int32); res.sy = np.empty(n, np.float64); res.sz = np.empty(n, np.float64)
            res.bin_start = np.empty(n_bins + 1, np.uint32); res.row_start = np.empty(self.n_rows + 1, np.int32)
            self._lib.oracle_get_grid(self._h, res.order.ctypes.data, res.sy.ctypes.data, res.sz.ctypes.data,
                                      res.bin_start.ctypes.data, res.row_start.ctypes.data)
        if "links" in want:
            def arr(cond):
                return np.empty(n, np.int32) if cond else None
            res.link_up_raw = arr(stage_mask & 2); res.link_dn_raw = arr(stage_mask & 2)
            res.link_up = arr(stage_mask & 4); res.link_dn = arr(stage_mask & 4)
            res.start_hit = np.empty(n_start, np.int32) if (stage_mask & 8) else None
            ptr = lambda a: a.ctypes.data if a is not None else None
            self._lib.oracle_get_links(self._h, ptr(res.link_up_raw), ptr(res.link_dn_raw), ptr(res.link_up),
                                       ptr(res.link_dn), ptr(res.start_hit))
        if "tracks" in want and (stage_mask & 16):
            res.x_ref = np.empty(n_trk); res.z_ref = np.empty(n_trk); res.chi2 = np.empty(n_trk)
            res.par = np.empty((n_trk, 5)); res.cov = np.empty((n_trk, 15))
            ints = np.empty((n_trk, 5), np.int32)
            res.hit_offset = np.empty(n_trk + 1, np.int32); res.hit_idx = np.empty(n_hit, np.int32)
            self._lib.oracle_get_tracks(self._h, res.x_ref.ctypes.data, res.z_ref.ctypes.data, res.par.ctypes.data,
                                        res.cov.ctypes.data, res.chi2.ctypes.data, ints.ctypes.data,
                                        res.hit_offset.ctypes.data, res.hit_idx.ctypes.data)
            res.n_hits, res.n_fit, res.first_row, res.last_row, res.trk_start_hit = (
                np.ascontiguousarray(ints[:, i]) for i in range(5))
        if "tracks" in want and (stage_mask & 32):
            res.owner = np.empty(n, np.int32); res.n_own = np.empty(n_trk, np.int32)
            res.selected = np.empty(int(self._lib.oracle_n_selected(self._h)), np.int32)
            self._lib.oracle_get_selection(self._h, res.owner.ctypes.data, res.n_own.ctypes.data, res.selected.ctypes.data)
        if "tracks" in want and (stage_mask & 64):
            res.res_trk = np.empty(n, np.int32); res.res_y = np.empty(n); res.res_z = np.empty(n)
            res.q_y = np.empty(n, np.int16); res.q_z = np.empty(n, np.int16)
            self._lib.oracle_get_residuals(self._h, res.res_trk.ctypes.data, res.res_y.ctypes.data, res.res_z.ctypes.data,
                                           res.q_y.ctypes.data, res.q_z.ctypes.data)
        return res

    # ---- unit entry points (pins) ---------------------------------------------------
    def kf_propagate(self, state, x2):
        st = np.ascontiguousarray(state, dtype=np.float64).copy()
        ok = self._lib.oracle_kf_propagate(self._h, st.ctypes.data_as(_dp), float(x2))
        return bool(ok), st

    def kf_update(self, state, ym, zm):
        st = np.ascontiguousarray(state, dtype=np.float64).copy()
        self._lib.oracle_kf_update(self._h, st.ctypes.data_as(_dp), float(ym), float(zm))
        return st

    def kf_dist2(self, state, ym, zm):
        st = np.ascontiguousarray(state, dtype=np.float64)
        return float(self._lib.oracle_kf_dist2(self._h, st.ctypes.data_as(_dp), float(ym), float(zm)))

    def kf_rotate(self, state, ca, sa):
        st = np.ascontiguousarray(state, dtype=np.float64).copy()
        ok = self._lib.oracle_kf_rotate(self._h, st.ctypes.data_as(_dp), float(ca), float(sa))
        return bool(ok), st

    def score(self, r, yc, zc, yu, zu, yd, zd):
        return float(self._lib.oracle_score(self._h, int(r), yc, zc, yu, zu, yd, zd))


@dataclasses.dataclass
class MergeResult:
    """S8 outputs of one sector: links per SELECTED track and the merged chains headed in the sector."""
    next_sec: np.ndarray = None
    next_trk: np.ndarray = None
    prev_sec: np.ndarray = None
    prev_trk: np.ndarray = None
    head: np.ndarray = None       # [n_merged] selected index of the lowest segment
    n_seg: np.ndarray = None
    n_hits: np.ndarray = None
    n_fit: np.ndarray = None
    first_row: np.ndarray = None
    last_row: np.ndarray = None
    frame_seg: np.ndarray = None  # segment (index in the chain) whose frame / z_ref the parameters are in
    x_ref: np.ndarray = None
    z_ref: np.ndarray = None
    par: np.ndarray = None
    cov: np.ndarray = None
    chi2: np.ndarray = None
    seg_offset: np.ndarray = None
    seg_sec: np.ndarray = None
    seg_trk: np.ndarray = None


def run_timeframe_merged(tf, precision="f32", sectors=None):
    """S1-S8 over a whole time frame: per-sector OracleResult (stage mask 0x7F) + MergeResult.  Keeps one oracle
    per sector alive for the cross-sector step."""
    lib = _load()
    ns = tf.n_sectors
    orcs = [Oracle(tf.params, precision) for _ in range(ns)]
    res = [orcs[s].run(tf.y[s], tf.z[s], tf.row[s], stage_mask=0x7F) for s in range(ns)]
    handles = (C.c_void_p * ns)(*[o._h for o in orcs])
    lib.oracle_merge(handles, ns)
    out = []
    for s in range(ns):
        k = int(res[s].selected.shape[0])
        m = MergeResult(next_sec=np.empty(k, np.int32), next_trk=np.empty(k, np.int32), prev_sec=np.empty(k, np.int32),
                        prev_trk=np.empty(k, np.int32))
        cnt = (C.c_int64 * 2)()
        lib.oracle_get_merge_links(orcs[s]._h, m.next_sec.ctypes.data, m.next_trk.ctypes.data, m.prev_sec.ctypes.data,
                                   m.prev_trk.ctypes.data, cnt)
        nm, nseg = int(cnt[0]), int(cnt[1])
        ints = np.empty((nm, 7), np.int32)
        m.x_ref = np.empty(nm); m.z_ref = np.empty(nm); m.chi2 = np.empty(nm); m.par = np.empty((nm, 5)); m.cov = np.empty((nm, 15))
        m.seg_offset = np.empty(nm + 1, np.int32); m.seg_sec = np.empty(nseg, np.int32); m.seg_trk = np.empty(nseg, np.int32)
        lib.oracle_get_merged(orcs[s]._h, ints.ctypes.data, m.x_ref.ctypes.data, m.z_ref.ctypes.data, m.par.ctypes.data,
                              m.cov.ctypes.data, m.chi2.ctypes.data, m.seg_offset.ctypes.data, m.seg_sec.ctypes.data,
                              m.seg_trk.ctypes.data)
        m.head, m.n_seg, m.n_hits, m.n_fit, m.first_row, m.last_row, m.frame_seg = (np.ascontiguousarray(ints[:, i]) for i in range(7))
        out.append(m)
    for o in orcs:
        o.close()
    return res, out


def merge_links_of_tables(params, sectors, precision="f32"):
    """S8 matching on hand-made selected tracks (pins of the match decisions).  `sectors`: per sector a list of dicts
    with first_row, last_row, x_ref, z_ref, par[5] and, for tracks that may be a lower segment, out = (x, p0..p4).
    Returns per sector (next_sec, next_trk, prev_sec, prev_trk)."""
    lib = _load()
    orcs = [Oracle(params, precision) for _ in sectors]
    for o, trks in zip(orcs, sectors):
        n = len(trks)
        ints = np.array([[t["first_row"], t["last_row"], 1 if t.get("out") is not None else 0] for t in trks], np.int32).reshape(n, 3)
        ref = np.array([[t["x_ref"], t["z_ref"]] for t in trks], np.float64).reshape(n, 2)
        par = np.array([t["par"] for t in trks], np.float64).reshape(n, 5)
        out = np.array([t["out"] if t.get("out") is not None else [0.0] * 6 for t in trks], np.float64).reshape(n, 6)
        lib.oracle_inject_selected(o._h, n, ints.ctypes.data, ref.ctypes.data, par.ctypes.data, out.ctypes.data)
    handles = (C.c_void_p * len(orcs))(*[o._h for o in orcs])
    lib.oracle_merge(handles, len(orcs))
    res = []
    for o, trks in zip(orcs, sectors):
        k = len(trks)
        a = [np.empty(k, np.int32) for _ in range(4)]
        cnt = (C.c_int64 * 2)()
        lib.oracle_get_merge_links(o._h, a[0].ctypes.data, a[1].ctypes.data, a[2].ctypes.data, a[3].ctypes.data, cnt)
        res.append(tuple(x.tolist() for x in a))
        o.close()
    return res


def select_tracks(n_clusters, hit_offset, hit_idx, max_shared_permille=500):
    """The S6 selector of the oracle on caller-given hit lists -> (owner, n_own, selected)."""
    lib = _load()
    ho = np.ascontiguousarray(hit_offset, dtype=np.int32)
    hi = np.ascontiguousarray(hit_idx, dtype=np.int32)
    nt = int(ho.shape[0]) - 1
    owner = np.empty(int(n_clusters), np.int32); n_own = np.empty(nt, np.int32); sel = np.empty(nt, np.int32)
    k = lib.oracle_select(int(n_clusters), nt, ho.ctypes.data, hi.ctypes.data, int(max_shared_permille),
                          owner.ctypes.data, n_own.ctypes.data, sel.ctypes.data)
    return owner, n_own, sel[:int(k)].copy()


def run_timeframe(tf, sectors=None, precision="f32", stage_mask=0x1F, brute=False):
    """Run the oracle over the sectors of a tpcsynth.Timeframe (independent units)."""
    orc = Oracle(tf.params, precision)
    out = {}
    for s in (range(tf.n_sectors) if sectors is None else sectors):
        out[s] = orc.run(tf.y[s], tf.z[s], tf.row[s], stage_mask=stage_mask, brute=brute)
    orc.close()
    return out
