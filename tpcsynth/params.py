"""Geometry, grid, window and cut tables of the TPC sector CA tracker (data, not code).

Source of every number: BASELINE.json:7 (pad-row layout, sigma, Bz = 0.5 T) and
SURVEY.md section 8(c) "Derived tables".  Tables are computed in double and then rounded
to fp32; both the CUDA library and the oracle consume the rounded values verbatim,
which is how two code-disjoint implementations stay bit-comparable.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

#: curvature per (q/pT): 0.299792458e-3 * Bz[kG] with Bz = 5 kG  [1/cm per 1/GeV]
BC_PER_QPT = 0.299792458e-3 * 5.0
#: drift velocity [cm/us] (BASELINE.json:9)
V_DRIFT = 2.58
#: LHC orbit [us]; 128 orbits = 11.38 ms (BASELINE.json:10)
ORBIT_US = 88.9244
#: half opening angle of a sector (20 degrees azimuth per sector)
TAN_HALF_SECTOR = math.tan(math.pi / 18.0)

N_ROWS_TPC = 152


def tpc_row_x() -> np.ndarray:
    """Pad-row radii (double): 63 rows at 0.75 cm from 85.225, 34 at 1.0, 30 at 1.2, 25 at 1.5.

    Reading G13: the first row of a region sits one *new* pitch after the last row of the
    previous region.
    """
    x = np.empty(N_ROWS_TPC, dtype=np.float64)
    x[0] = 85.225
    for i in range(1, N_ROWS_TPC):
        x[i] = x[i - 1] + row_pitch(i)
    return x


def row_pitch(i: int) -> float:
    if i < 63:
        return 0.75
    if i < 97:
        return 1.0
    if i < 127:
        return 1.2
    return 1.5


@dataclasses.dataclass
class TrackerParams:
    """All tables the tracker needs.  Float tables hold fp32-representable values."""
    n_sectors: int
    n_rows: int
    row_x: np.ndarray            # [n_rows] f32
    grid_y_lo: np.ndarray        # [n_rows] f32
    grid_inv_bin_y: np.ndarray   # [n_rows] f32
    grid_ny: np.ndarray          # [n_rows] i32
    grid_z_lo: float
    grid_inv_bin_z: np.ndarray   # [n_rows] f32
    grid_nz: np.ndarray          # [n_rows] i32
    nf_hy_up: np.ndarray         # [n_rows] f32  S2 window half-widths
    nf_hz_up: np.ndarray
    nf_hy_dn: np.ndarray
    nf_hz_dn: np.ndarray
    nf_cut: np.ndarray           # [n_rows] f32  S2 score cut
    kappa_per_qpt: float
    err2_y: float
    err2_z: float
    init_cov: np.ndarray         # [5] f32
    tc_win_y: float
    tc_win_z: float
    tc_gate: float
    max_sinphi: float
    grid_margin: float
    tc_max_gap: int
    tc_min_hits: int
    sel_max_shared_permille: int = 500   # S6 selector: a tracklet survives iff at most this share of its hits is not its own
    res_inv_quantum: float = 128.0       # S7 residual front end: residuals are quantised to round(res * this) (1/128 cm)
    # S8 cross-sector merging: neighbour relation (18 sectors per side, 20 degrees apart) and match windows
    sectors_per_side: int = 18
    sector_cos: float = float(np.float32(math.cos(math.pi / 9.0)))
    sector_sin: float = float(np.float32(math.sin(math.pi / 9.0)))
    mg_max_row_gap: int = 8
    mg_dy: float = 1.0
    mg_dz: float = 1.0
    mg_dsin: float = 0.05
    mg_zpre: float = 32.0
    # informative (not consumed by the tracker)
    sigma: float = 0.1
    z_hi: float = 250.0
    bin_size: np.ndarray | None = None

    def bins_per_sector(self) -> int:
        return int(np.sum(self.grid_ny.astype(np.int64) * self.grid_nz.astype(np.int64)))

    def copy(self, **kw) -> "TrackerParams":
        d = {f.name: getattr(self, f.name) for f in dataclasses.fields(self)}
        for k, v in d.items():
            if isinstance(v, np.ndarray):
                d[k] = v.copy()
        d.update(kw)
        return TrackerParams(**d)


def _f32(a):
    return np.asarray(a, dtype=np.float64).astype(np.float32)


def default_params(n_sectors: int = 36, sigma: float = 0.1, z_hi: float = 250.0,
                   row_x: np.ndarray | None = None, pitch: np.ndarray | None = None,
                   bin_scale: float = 1.0, grid_margin: float = 0.01,
                   nf_slope: float = 2.0) -> TrackerParams:
    """SURVEY.md 8(c) 'Derived tables'.

    `row_x`/`pitch` may be overridden (geometry is data: the dyadic test geometry of pin
    P4 uses it); `bin_scale` scales the grid bin size (metamorphic pin P3: links must not
    depend on it); `z_hi` is the upper end of the z axis the tracker sees
    (250 + v_drift * T for a time frame).
    """
    if row_x is None:
        row_x = tpc_row_x()
        pitch = np.array([row_pitch(i) for i in range(N_ROWS_TPC)], dtype=np.float64)
    row_x = np.asarray(row_x, dtype=np.float64)
    n_rows = row_x.shape[0]
    if pitch is None:
        pitch = np.empty(n_rows)
        pitch[1:] = np.diff(row_x)
        pitch[0] = pitch[1]
    nf_pad = 5.0 * sigma
    dxu = np.empty(n_rows)
    dxd = np.empty(n_rows)
    dxu[:-1] = np.diff(row_x)
    dxu[-1] = dxu[-2]
    dxd[1:] = np.diff(row_x)
    dxd[0] = dxd[1]
    ymax = row_x * TAN_HALF_SECTOR
    h_up = nf_slope * dxu + nf_pad
    h_dn = nf_slope * dxd + nf_pad
    nf_cut = 16.0 * sigma * sigma * (dxd ** 2 + (dxu + dxd) ** 2 + dxu ** 2)
    bin_sz = 2.0 * (nf_slope * pitch + nf_pad) * bin_scale
    grid_y_lo = -(ymax + 1.0)
    grid_ny = np.ceil(2.0 * (ymax + 1.0) / bin_sz).astype(np.int32)
    grid_nz = np.ceil((z_hi + 2.0) / bin_sz).astype(np.int32)
    return TrackerParams(
        n_sectors=int(n_sectors), n_rows=int(n_rows),
        row_x=_f32(row_x),
        grid_y_lo=_f32(grid_y_lo), grid_inv_bin_y=_f32(1.0 / bin_sz), grid_ny=grid_ny,
        grid_z_lo=float(np.float32(-1.0)), grid_inv_bin_z=_f32(1.0 / bin_sz), grid_nz=grid_nz,
        nf_hy_up=_f32(h_up), nf_hz_up=_f32(h_up), nf_hy_dn=_f32(h_dn), nf_hz_dn=_f32(h_dn),
        nf_cut=_f32(nf_cut),
        kappa_per_qpt=float(np.float32(BC_PER_QPT)),
        err2_y=float(np.float32(sigma * sigma)), err2_z=float(np.float32(sigma * sigma)),
        init_cov=_f32([1.0, 1.0, 0.25, 1.0, 25.0]),
        tc_win_y=3.0, tc_win_z=3.0, tc_gate=20.0,
        max_sinphi=float(np.float32(0.95)), grid_margin=float(np.float32(grid_margin)),
        tc_max_gap=4, tc_min_hits=10,
        sigma=float(sigma), z_hi=float(z_hi), bin_size=bin_sz,
    )
