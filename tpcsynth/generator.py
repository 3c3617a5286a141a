"""Seeded synthetic ALICE-TPC-shaped cluster generator (BASELINE.json:7-11, configs 0-4).

The recipe (readings G1-G13 of SURVEY.md section 8(c), restated in DESIGN.md):

* primary helix tracks from (0, 0, z_v) in a uniform Bz = 0.5 T, exact circles, no
  scattering; radius R = pT / Bc, turning sense h = +-1 equiprobable;
* local sector frame: x radial through the sector centre alpha_s = (s + 0.5) * 20 deg,
  pad rows are the planes x = row_x[i]; a crossing belongs to the sector in which
  |y| <= x * tan(10 deg); per (track, row) the crossing with the smallest arc angle
  theta < pi is kept (outgoing leg only; loopers end at r = 2R);
* z_true = z_v + sinh(eta) * R * theta, kept if |z_true| <= 250; z >= 0 -> sectors 0..17
  (A side), z < 0 -> sectors 18..35 (C side); the tracker receives
  z = |z_true| + v_drift * t_collision;
* Gaussian smearing of y and z, independent per-(track,row) drop-out, uniform noise
  clusters (fraction of the signal count per sector), Moyal ("Landau-like") charge;
* time frames: Poisson number of collisions, uniform times, impact-parameter law for the
  multiplicity.

All geometry here is double precision and lives OUTSIDE the tracking pipeline, so libm
transcendentals are fine.  Random numbers: numpy Philox streams keyed by
(seed, config, collision | sector), so the output does not depend on evaluation order.
"""
from __future__ import annotations

import dataclasses
import math
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from .params import (BC_PER_QPT, ORBIT_US, TAN_HALF_SECTOR, V_DRIFT, TrackerParams,
                     default_params, tpc_row_x)

BASE_SEED = 220807412
SECTOR_ANGLE = math.radians(20.0)

#: BASELINE.json:7-11.  n_orbits = 0 means "one collision at t = 0".
CONFIGS = {
    0: dict(name="single-sector-100", n_sectors=1, n_orbits=0, n_tracks=100, inv_pt=(0.2, 5.0),
            sigma=0.1, drop=0.02, noise=0.05, zv_sigma=0.0, fold_eta=True),
    1: dict(name="central-PbPb-10k", n_sectors=36, n_orbits=0, n_tracks=10000, inv_pt=(0.15, 6.7),
            sigma=0.1, drop=0.02, noise=0.05, zv_sigma=5.0, fold_eta=False),
    2: dict(name="tf-32-orbits", n_sectors=36, n_orbits=32, n_tracks=None, inv_pt=(0.15, 6.7),
            sigma=0.1, drop=0.02, noise=0.05, zv_sigma=5.0, fold_eta=False),
    3: dict(name="tf-128-orbits", n_sectors=36, n_orbits=128, n_tracks=None, inv_pt=(0.15, 6.7),
            sigma=0.1, drop=0.02, noise=0.05, zv_sigma=5.0, fold_eta=False),
    4: dict(name="lowpt-stress-15k", n_sectors=36, n_orbits=0, n_tracks=15000, inv_pt=(0.1, 10.0),
            sigma=0.2, drop=0.10, noise=0.20, zv_sigma=5.0, fold_eta=False),
}


@dataclasses.dataclass
class Timeframe:
    """Clusters per sector (shuffled, SoA) + generator truth."""
    config: int
    seed: int
    params: TrackerParams
    x: list      # per sector f32[n]
    y: list
    z: list
    q: list
    row: list    # per sector u16[n]
    label: list  # per sector i32[n]: global track id, -1 = noise
    # per-track truth (global track id = index)
    trk_coll: np.ndarray
    trk_h: np.ndarray
    trk_pt: np.ndarray
    trk_phi0: np.ndarray
    trk_eta: np.ndarray
    trk_zv: np.ndarray
    coll_t: np.ndarray   # [n_coll] us

    @property
    def n_sectors(self) -> int:
        return len(self.y)

    @property
    def n_clusters(self) -> int:
        return int(sum(a.shape[0] for a in self.y))

    def sector_counts(self) -> np.ndarray:
        return np.array([a.shape[0] for a in self.y], dtype=np.int64)


def _rng(*key) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(np.random.SeedSequence([int(k) for k in key])))


def _moyal(rng, n):
    g = rng.standard_normal(n)
    q = 50.0 - 10.0 * np.log(g * g + 1e-300)
    return np.maximum(q, 1.0).astype(np.float32)


def _collision_clusters(row_x, h, pt, phi0, eta, zv, t_us, sigma, drop, rng, single_sector):
    """Clusters of one collision.  Returns (sector u8, row u8, y f32, z f32, track i32)."""
    nt = h.shape[0]
    nr = row_x.shape[0]
    R = (pt / BC_PER_QPT)[:, None]
    hh = h[:, None]
    cx = (-h * (pt / BC_PER_QPT) * np.sin(phi0))[:, None]
    cy = (h * (pt / BC_PER_QPT) * np.cos(phi0))[:, None]
    xr = row_x[None, :]
    # sector guess from the azimuth of the track at radius row_x (circle through the origin)
    ratio = xr / (2.0 * R)
    reach = ratio < 1.0
    thg = 2.0 * np.arcsin(np.minimum(ratio, 1.0))
    az = phi0[:, None] + hh * thg * 0.5
    s0 = np.floor(az / SECTOR_ANGLE).astype(np.int64)
    best_th = np.full((nt, nr), np.inf)
    best_y = np.zeros((nt, nr))
    best_s = np.zeros((nt, nr), dtype=np.int64)
    ymax = xr * TAN_HALF_SECTOR
    for k in (-1, 0, 1):
        s = np.mod(s0 + k, 18)
        alpha = (s + 0.5) * SECTOR_ANGLE
        ca, sa = np.cos(alpha), np.sin(alpha)
        Xc = cx * ca + cy * sa
        Yc = -cx * sa + cy * ca
        disc = R * R - (xr - Xc) ** 2
        ok0 = reach & (disc >= 0.0)
        sq = np.sqrt(np.maximum(disc, 0.0))
        psi0 = np.arctan2(-Yc, -Xc)
        for sgn in (-1.0, 1.0):
            yy = Yc + sgn * sq
            th = np.mod(hh * (np.arctan2(yy - Yc, xr - Xc) - psi0), 2.0 * math.pi)
            ok = ok0 & (th < math.pi) & (np.abs(yy) <= ymax) & (th < best_th)
            best_th = np.where(ok, th, best_th)
            best_y = np.where(ok, yy, best_y)
            best_s = np.where(ok, s, best_s)
    keep = np.isfinite(best_th)
    th = np.where(keep, best_th, 0.0)
    z_true = zv[:, None] + np.sinh(eta)[:, None] * R * th
    keep &= np.abs(z_true) <= 250.0
    # random draws have fixed shapes so that the stream does not depend on the masks
    u_drop = rng.random((nt, nr))
    gy = rng.standard_normal((nt, nr))
    gz = rng.standard_normal((nt, nr))
    keep &= u_drop >= drop
    side = (z_true < 0.0).astype(np.int64)
    sector = best_s + 18 * side
    if single_sector:
        keep &= sector == 0
    z_loc = np.abs(z_true) + V_DRIFT * t_us + sigma * gz
    y_loc = best_y + sigma * gy
    ti, ri = np.nonzero(keep)
    return (sector[ti, ri].astype(np.uint8), ri.astype(np.uint8),
            y_loc[ti, ri].astype(np.float32), z_loc[ti, ri].astype(np.float32),
            ti.astype(np.int32))


def generate(config: int, seed: int | None = None, mult_scale: float = 1.0,
             n_tracks: int | None = None, n_orbits: int | None = None,
             threads: int | None = None, noise: float | None = None,
             drop: float | None = None, sigma: float | None = None,
             coll_times=None, coll_mult=None) -> Timeframe:
    """Generate the clusters of BASELINE.json config `config` (0..4).

    `mult_scale` scales the per-collision multiplicity (config 3 at 2.75
    reaches the ~4e8 clusters BASELINE.json:10 names); `n_tracks` / `n_orbits` / `noise` /
    `drop` / `sigma` override the config for reduced-size test variants; `coll_times` [us] (with
    `coll_mult` tracks each, default n_tracks or 500) replaces the Poisson / impact-parameter draw of a
    time-frame config by a hand-placed list of collisions (the z axis keeps the config's full length).
    """
    cfg = dict(CONFIGS[config])
    if seed is None:
        seed = BASE_SEED + config
    if n_tracks is not None:
        cfg["n_tracks"] = n_tracks
    if n_orbits is not None:
        cfg["n_orbits"] = n_orbits
    if noise is not None:
        cfg["noise"] = noise
    if drop is not None:
        cfg["drop"] = drop
    if sigma is not None:
        cfg["sigma"] = sigma
    sigma = cfg["sigma"]
    n_sectors = cfg["n_sectors"]
    row_x = tpc_row_x()
    nr = row_x.shape[0]

    # ---- collisions ----
    rng0 = _rng(seed, config, 0)
    if cfg["n_orbits"] > 0:
        T = cfg["n_orbits"] * ORBIT_US
        n_coll = int(rng0.poisson(50e3 * T * 1e-6))
        coll_t = rng0.random(n_coll) * T
        b = 15.0 * np.sqrt(rng0.random(n_coll))
        mult = np.rint(10000.0 * (1.0 - b / 15.0) ** 2 * mult_scale).astype(np.int64)
        if coll_times is not None:
            coll_t = np.asarray(coll_times, dtype=np.float64)
            assert coll_t.ndim == 1 and np.all(coll_t >= 0.0) and np.all(coll_t <= T)
            n_coll = int(coll_t.shape[0])
            if coll_mult is None:
                coll_mult = cfg["n_tracks"] or 500
            mult = np.broadcast_to(np.asarray(coll_mult, dtype=np.int64), (n_coll,)).copy()
    else:
        T = 0.0
        n_coll = 1
        coll_t = np.zeros(1)
        mult = np.array([int(round(cfg["n_tracks"] * mult_scale))], dtype=np.int64)
    z_hi = 250.0 + V_DRIFT * T
    params = default_params(n_sectors=n_sectors, sigma=sigma, z_hi=z_hi)
    trk_off = np.concatenate([[0], np.cumsum(mult)])
    n_trk = int(trk_off[-1])

    trk_h = np.empty(n_trk, dtype=np.int8)
    trk_pt = np.empty(n_trk)
    trk_phi0 = np.empty(n_trk)
    trk_eta = np.empty(n_trk)
    trk_zv = np.empty(n_trk)
    trk_coll = np.repeat(np.arange(n_coll, dtype=np.int32), mult)

    def one(c):
        nt = int(mult[c])
        rng = _rng(seed, config, 1, c)
        h = np.where(rng.random(nt) < 0.5, -1.0, 1.0)
        inv_pt = rng.uniform(cfg["inv_pt"][0], cfg["inv_pt"][1], nt)
        if cfg["fold_eta"]:
            phi0 = rng.uniform(0.0, SECTOR_ANGLE, nt)     # sector 0 spans [0, 20 deg]
        else:
            phi0 = rng.uniform(0.0, 2.0 * math.pi, nt)
        eta = rng.uniform(-0.9, 0.9, nt)
        if cfg["fold_eta"]:
            eta = np.abs(eta)
        zv = rng.standard_normal(nt) * cfg["zv_sigma"]
        pt = 1.0 / inv_pt
        o = int(trk_off[c])
        trk_h[o:o + nt] = h
        trk_pt[o:o + nt] = pt
        trk_phi0[o:o + nt] = phi0
        trk_eta[o:o + nt] = eta
        trk_zv[o:o + nt] = zv
        if nt == 0:
            e = np.empty(0)
            return (e.astype(np.uint8), e.astype(np.uint8), e.astype(np.float32),
                    e.astype(np.float32), e.astype(np.int32))
        sec, row, y, z, ti = _collision_clusters(row_x, h, pt, phi0, eta, zv, float(coll_t[c]),
                                                 sigma, cfg["drop"], rng, cfg["fold_eta"])
        return sec, row, y, z, (ti + o).astype(np.int32)

    if threads is None:
        threads = min(16, len(os.sched_getaffinity(0)))
    if n_coll > 1 and threads > 1:
        with ThreadPoolExecutor(threads) as ex:
            parts = list(ex.map(one, range(n_coll)))
    else:
        parts = [one(c) for c in range(n_coll)]
    if not parts:       # a Poisson draw of zero collisions: an empty time frame is a legal input (reading N8)
        e = np.empty(0)
        parts = [(e.astype(np.uint8), e.astype(np.uint8), e.astype(np.float32), e.astype(np.float32), e.astype(np.int32))]
    sec = np.concatenate([p[0] for p in parts])
    row = np.concatenate([p[1] for p in parts])
    y = np.concatenate([p[2] for p in parts])
    z = np.concatenate([p[3] for p in parts])
    lab = np.concatenate([p[4] for p in parts])
    del parts

    # ---- split per sector, add noise, shuffle ----
    counts = np.bincount(sec, minlength=n_sectors)[:n_sectors]
    idx = np.argsort(sec, kind="stable")
    starts = np.concatenate([[0], np.cumsum(counts)])
    row_x32 = params.row_x
    ymax = tpc_row_x() * TAN_HALF_SECTOR
    X, Y, Z, Q, ROW, LAB = [], [], [], [], [], []

    def finish(s):
        sl = idx[starts[s]:starts[s + 1]]
        rng = _rng(seed, config, 2, s)
        n_sig = sl.shape[0]
        n_noise = int(round(cfg["noise"] * n_sig))
        nrow = rng.integers(0, nr, n_noise)
        ny = (rng.random(n_noise) * 2.0 - 1.0) * ymax[nrow]
        nz = rng.random(n_noise) * z_hi
        r_all = np.concatenate([row[sl].astype(np.uint16), nrow.astype(np.uint16)])
        y_all = np.concatenate([y[sl], ny.astype(np.float32)])
        z_all = np.concatenate([z[sl], nz.astype(np.float32)])
        l_all = np.concatenate([lab[sl], np.full(n_noise, -1, dtype=np.int32)])
        q_all = _moyal(rng, n_sig + n_noise)
        perm = rng.permutation(n_sig + n_noise)
        r_all = r_all[perm]
        return (row_x32[r_all], y_all[perm], z_all[perm], q_all[perm], r_all, l_all[perm])

    if n_sectors > 1 and threads > 1:
        with ThreadPoolExecutor(threads) as ex:
            outs = list(ex.map(finish, range(n_sectors)))
    else:
        outs = [finish(s) for s in range(n_sectors)]
    for o in outs:
        X.append(o[0]); Y.append(o[1]); Z.append(o[2]); Q.append(o[3]); ROW.append(o[4]); LAB.append(o[5])
    return Timeframe(config=config, seed=seed, params=params, x=X, y=Y, z=Z, q=Q, row=ROW, label=LAB,
                     trk_coll=trk_coll, trk_h=trk_h, trk_pt=trk_pt, trk_phi0=trk_phi0,
                     trk_eta=trk_eta, trk_zv=trk_zv, coll_t=coll_t)


def truth_state(tf: Timeframe, track: int, sector: int, x: float):
    """Generator-truth local state (y, z, sin phi, dz/ds, q/pT-like p4) of `track` at the
    plane `x` of `sector` (double precision; used by the statistical pins P6/P8).

    p4 is the *local* signed curvature over Bc (d sin(phi)/dx = Bc * p4), so no charge or
    field sign convention enters (reading G2).  Returns None if the circle does not reach x.
    """
    h = float(tf.trk_h[track]); pt = float(tf.trk_pt[track])
    phi0 = float(tf.trk_phi0[track]); eta = float(tf.trk_eta[track]); zv = float(tf.trk_zv[track])
    t = float(tf.coll_t[tf.trk_coll[track]])
    R = pt / BC_PER_QPT
    cx, cy = -h * R * math.sin(phi0), h * R * math.cos(phi0)
    s18 = sector % 18
    alpha = (s18 + 0.5) * SECTOR_ANGLE
    Xc = cx * math.cos(alpha) + cy * math.sin(alpha)
    Yc = -cx * math.sin(alpha) + cy * math.cos(alpha)
    disc = R * R - (x - Xc) ** 2
    if disc < 0:
        return None
    psi0 = math.atan2(-Yc, -Xc)
    best = None
    for sgn in (-1.0, 1.0):
        yy = Yc + sgn * math.sqrt(disc)
        th = (h * (math.atan2(yy - Yc, x - Xc) - psi0)) % (2.0 * math.pi)
        if th < math.pi and (best is None or th < best[0]):
            best = (th, yy)
    if best is None:
        return None
    th, yy = best
    z_true = zv + math.sinh(eta) * R * th
    zsign = -1.0 if (sector >= 18) else 1.0
    sinphi = h * (x - Xc) / R
    return dict(y=yy, z=zsign * z_true + V_DRIFT * t, sinphi=sinphi,
                dzds=zsign * math.sinh(eta), p4=h / pt)


# ----------------------------------------------------------------------------------------
# Noise-free fixtures for the pins (inputs only: circle / line geometry in double precision)
# ----------------------------------------------------------------------------------------

def straight_tracks(row_x, y0, ty, z0, tz):
    """Noise-free straight lines y = y0 + ty*(x - row_x[0]), z = z0 + tz*(x - row_x[0]).

    Returns per-cluster (row u16, y f64, z f64, track i32), one cluster per (track, row).
    """
    row_x = np.asarray(row_x, dtype=np.float64)
    y0, ty, z0, tz = (np.atleast_1d(np.asarray(a, dtype=np.float64)) for a in (y0, ty, z0, tz))
    dx = row_x[None, :] - row_x[0]
    y = y0[:, None] + ty[:, None] * dx
    z = z0[:, None] + tz[:, None] * dx
    nt, nr = y.shape
    row = np.tile(np.arange(nr, dtype=np.uint16), nt)
    trk = np.repeat(np.arange(nt, dtype=np.int32), nr)
    return row, y.ravel(), z.ravel(), trk


def helix_hits(row_x, x0, y0, z0, sinphi0, dzds, kappa):
    """Exact noise-free helix in the local frame, double precision.

    sin(phi)(x) = sinphi0 + kappa*(x - x0); y(x) = y0 + (cos(phi0) - cos(phi(x)))/kappa;
    arc length s(x) = (phi(x) - phi0)/kappa; z = z0 + dzds*s.  Rows the circle does not
    reach (|sin phi| >= 1) are dropped.  Returns (rows, y, z, sinphi) as f64 arrays.
    """
    row_x = np.asarray(row_x, dtype=np.float64)
    sp = sinphi0 + kappa * (row_x - x0)
    ok = np.abs(sp) < 1.0
    rows = np.nonzero(ok)[0]
    sp = sp[ok]
    xs = row_x[ok]
    cp0 = math.sqrt(1.0 - sinphi0 * sinphi0)
    cp = np.sqrt(1.0 - sp * sp)
    if abs(kappa) > 1e-14:
        y = y0 + (cp0 - cp) / kappa
        s = (np.arcsin(sp) - math.asin(sinphi0)) / kappa
    else:
        y = y0 + (xs - x0) * sinphi0 / cp0
        s = (xs - x0) / cp0
    z = z0 + dzds * s
    return rows.astype(np.int64), y, z, sp
