"""Element-by-element comparison of the CUDA path (paper_2208_07412_b200.SectorOutput) with the
CPU oracle (oracle.OracleResult).  Used by the -m gpu parity tests, smoke() and bench.py's check.

The bar (BASELINE.json:5 north_star, readings N4/N5 of DESIGN.md 3.8):
  * grid, links, start hits, track membership: bit-exact.  Link exception: clusters whose link pair
    differs are allowed iff the oracle-rescored scores of the two pairs agree to 1e-5 relative,
    and such clusters are <= 0.1 % of the oracle's linked clusters;
  * fitted parameters: |a-b| <= 1e-4 * max(|a|,|b|,floor_i), floors (1 cm, 1 cm, 0.1, 0.1, 0.1/GeV);
    covariances: |dC_ij| <= 1e-4 * sqrt(C_ii C_jj); chi2: 1e-4 relative (floor 1e-3).
"""
from __future__ import annotations

import numpy as np

PAR_FLOOR = np.array([1.0, 1.0, 0.1, 0.1, 0.1])
TRI = [(i, j) for i in range(5) for j in range(i + 1)]   # k = i(i+1)/2 + j


class ParityError(AssertionError):
    pass


def _eq(name, a, b, report):
    a = np.asarray(a); b = np.asarray(b)
    if a.shape != b.shape:
        raise ParityError(f"{name}: shape {a.shape} (gpu) vs {b.shape} (oracle)")
    if not np.array_equal(a, b):
        bad = np.nonzero(a != b)[0]
        raise ParityError(f"{name}: {bad.size} of {a.size} differ; first at {bad[0]}: gpu {a[bad[0]]} oracle {b[bad[0]]}")
    report[name] = "bit-exact"


def compare_sector(gpu, orc, oracle_obj=None, srow=None, stages=0x1F) -> dict:
    """Raise ParityError on any violation of the bar; return a small report dict."""
    rep = {}
    if gpu.n != orc.n:
        raise ParityError(f"n_clusters {gpu.n} vs {orc.n}")
    if stages & 1:
        _eq("order", gpu.order, orc.order, rep)
        _eq("sy", gpu.sy, orc.sy.astype(np.float32), rep)
        _eq("sz", gpu.sz, orc.sz.astype(np.float32), rep)
        _eq("bin_start", gpu.bin_start, orc.bin_start, rep)
        _eq("row_start", gpu.row_start, orc.row_start, rep)
    if stages & 2:
        du = gpu.link_up_raw != orc.link_up_raw
        dd = gpu.link_dn_raw != orc.link_dn_raw
        diff = np.nonzero(du | dd)[0]
        rep["links_differing"] = int(diff.size)
        if diff.size:
            # reading N4: rescore both pairs with the oracle's arithmetic
            if oracle_obj is None or srow is None:
                raise ParityError(f"raw links differ at {diff.size} clusters (first {diff[0]})")
            n_linked = max(int((orc.link_up_raw >= 0).sum()), 1)
            for c in diff:
                gu, gd, ou, od = gpu.link_up_raw[c], gpu.link_dn_raw[c], orc.link_up_raw[c], orc.link_dn_raw[c]
                if min(gu, gd, ou, od) < 0:
                    raise ParityError(f"raw link of cluster {c}: gpu ({gu},{gd}) oracle ({ou},{od})")
                r = int(srow[c])
                sg = oracle_obj.score(r, orc.sy[c], orc.sz[c], orc.sy[gu], orc.sz[gu], orc.sy[gd], orc.sz[gd])
                so = oracle_obj.score(r, orc.sy[c], orc.sz[c], orc.sy[ou], orc.sz[ou], orc.sy[od], orc.sz[od])
                if abs(sg - so) > 1e-5 * max(sg, so, 1e-12):
                    raise ParityError(f"raw link of cluster {c}: scores {sg} (gpu pair) vs {so} (oracle pair)")
            if diff.size > 1e-3 * n_linked:
                raise ParityError(f"{diff.size} differing links > 0.1 % of {n_linked}")
        else:
            rep["link_up_raw"] = rep["link_dn_raw"] = "bit-exact"
    if stages & 4:
        _eq("link_up", gpu.link_up, orc.link_up, rep)
        _eq("link_dn", gpu.link_dn, orc.link_dn, rep)
    if stages & 8:
        _eq("start_hit", gpu.start_hit, orc.start_hit, rep)
    if stages & 16:
        if gpu.n_tracks != orc.n_tracks:
            raise ParityError(f"n_tracks {gpu.n_tracks} (gpu) vs {orc.n_tracks} (oracle)")
        _eq("trk_start_hit", gpu.trk_start_hit, orc.trk_start_hit, rep)
        _eq("n_hits", gpu.n_hits, orc.n_hits, rep)
        _eq("hit_offset", gpu.hit_offset, orc.hit_offset, rep)
        _eq("hit_idx", gpu.hit_idx, orc.hit_idx, rep)
        _eq("n_fit", gpu.n_fit, orc.n_fit, rep)
        _eq("first_row", gpu.first_row, orc.first_row, rep)
        _eq("last_row", gpu.last_row, orc.last_row, rep)
        _eq("x_ref", gpu.x_ref, orc.x_ref.astype(np.float32), rep)
        _eq("z_ref", gpu.z_ref, orc.z_ref.astype(np.float32), rep)
        if orc.n_tracks:
            gp = gpu.par.astype(np.float64); op = orc.par
            tol = 1e-4 * np.maximum(np.maximum(np.abs(gp), np.abs(op)), PAR_FLOOR[None, :])
            bad = np.abs(gp - op) > tol
            if bad.any():
                t, i = np.argwhere(bad)[0]
                raise ParityError(f"par[{t},{i}]: gpu {gp[t, i]} oracle {op[t, i]}")
            gc = gpu.cov.astype(np.float64); oc = orc.cov
            diag = np.stack([oc[:, i * (i + 1) // 2 + i] for i in range(5)], axis=1)
            for k, (i, j) in enumerate(TRI):
                lim = 1e-4 * np.sqrt(np.abs(diag[:, i] * diag[:, j]))
                b = np.abs(gc[:, k] - oc[:, k]) > lim
                if b.any():
                    t = np.nonzero(b)[0][0]
                    raise ParityError(f"cov[{t},{k}]: gpu {gc[t, k]} oracle {oc[t, k]}")
            g2 = gpu.chi2.astype(np.float64)
            b = np.abs(g2 - orc.chi2) > 1e-4 * np.maximum(np.maximum(np.abs(g2), np.abs(orc.chi2)), 1e-3)
            if b.any():
                t = np.nonzero(b)[0][0]
                raise ParityError(f"chi2[{t}]: gpu {g2[t]} oracle {orc.chi2[t]}")
            rep["par_bit_exact"] = bool(np.array_equal(gpu.par, op.astype(np.float32)))
            rep["cov_bit_exact"] = bool(np.array_equal(gpu.cov, oc.astype(np.float32)))
            rep["chi2_bit_exact"] = bool(np.array_equal(gpu.chi2, orc.chi2.astype(np.float32)))
        rep["n_tracks"] = int(orc.n_tracks)
    return rep


def compare_timeframe(tracker, tf, oracle_obj, sectors=None, stages=0x1F) -> dict:
    """Compare every (or the given) sector of an already-run Tracker against the oracle."""
    tot = dict(sectors=0, n_clusters=0, n_tracks=0, links_differing=0, par_bit_exact=True, cov_bit_exact=True)
    for s in (range(tf.n_sectors) if sectors is None else sectors):
        g = tracker.get_tracks(s)
        o = oracle_obj.run(tf.y[s], tf.z[s], tf.row[s], stage_mask=stages)
        srow = tf.row[s][o.order] if o.order is not None else None
        try:
            rep = compare_sector(g, o, oracle_obj, srow, stages)
        except ParityError as e:
            raise ParityError(f"sector {s}: {e}") from None
        tot["sectors"] += 1
        tot["n_clusters"] += o.n
        tot["n_tracks"] += rep.get("n_tracks", 0)
        tot["links_differing"] += rep.get("links_differing", 0)
        tot["par_bit_exact"] &= rep.get("par_bit_exact", True)
        tot["cov_bit_exact"] &= rep.get("cov_bit_exact", True)
    return tot


def compare_selection(tracker, tf, oracle_obj, sectors=None) -> dict:
    """S6 (tracklet selector): owner / n_own / selected bit-exact against the oracle; the compact table of the
    selected tracks must be the S5 table gathered at `selected` (bit-exact, hit lists included)."""
    from paper_2208_07412_b200 import binding as B
    tot = dict(sectors=0, n_tracks=0, n_selected=0)
    for s in (range(tf.n_sectors) if sectors is None else sectors):
        o = oracle_obj.run(tf.y[s], tf.z[s], tf.row[s], stage_mask=0x3F)
        g = tracker.get_tracks(s, B.OUT_TRACKS | B.OUT_SELECTION)
        c = tracker.get_tracks(s, B.OUT_TRACKS_SEL)
        rep = {}
        try:
            _eq("owner", g.owner, o.owner, rep)
            _eq("n_own", g.n_own, o.n_own, rep)
            _eq("selected", g.selected, o.selected, rep)
            sel = o.selected
            for f in ("x_ref", "z_ref", "chi2", "par", "cov", "n_hits", "n_fit", "first_row", "last_row", "trk_start_hit"):
                _eq("sel." + f, getattr(c, f), getattr(g, f)[sel], rep)
            off = np.concatenate([[0], np.cumsum(o.n_hits[sel])]).astype(np.int32)
            _eq("sel.hit_offset", c.hit_offset, off, rep)
            idx = (np.concatenate([o.hit_idx[o.hit_offset[t]:o.hit_offset[t + 1]] for t in sel]) if len(sel)
                   else np.empty(0, np.int32))
            _eq("sel.hit_idx", c.hit_idx, idx, rep)
        except ParityError as e:
            raise ParityError(f"sector {s}: {e}") from None
        tot["sectors"] += 1; tot["n_tracks"] += int(o.n_tracks); tot["n_selected"] += int(len(o.selected))
    return tot


def compare_residuals(tracker, tf, oracle_obj, sectors=None) -> dict:
    """S7 (track-residual front end): res_trk and the quantised residuals bit-exact (integers), the fp32
    residuals bit-exact as well (same operation order; the bar would allow 1e-4 relative)."""
    from paper_2208_07412_b200 import binding as B
    tot = dict(sectors=0, n_clusters=0, n_attached=0)
    for s in (range(tf.n_sectors) if sectors is None else sectors):
        o = oracle_obj.run(tf.y[s], tf.z[s], tf.row[s], stage_mask=0x7F)
        g = tracker.get_tracks(s, B.OUT_RESIDUALS)
        rep = {}
        try:
            _eq("res_trk", g.res_trk, o.res_trk, rep)
            _eq("q_y", g.q_y, o.q_y, rep)
            _eq("q_z", g.q_z, o.q_z, rep)
            _eq("res_y", g.res_y, o.res_y.astype(np.float32), rep)
            _eq("res_z", g.res_z, o.res_z.astype(np.float32), rep)
        except ParityError as e:
            raise ParityError(f"sector {s}: {e}") from None
        tot["sectors"] += 1; tot["n_clusters"] += int(o.n); tot["n_attached"] += int((o.res_trk >= 0).sum())
    return tot


def compare_merge(tracker, tf, precision="f32") -> dict:
    """S8 (cross-sector merging + chain refit): the links per selected track bit-exact; per chain head the segment
    count, hit counts, rows, reference plane bit-exact and the refitted parameters / covariance / chi2 within the
    1e-4 bar of N5 (same operation order: observed bit-exact is reported)."""
    from oracle import run_timeframe_merged
    from paper_2208_07412_b200 import binding as B
    res, mg = run_timeframe_merged(tf, precision)
    tot = dict(sectors=0, n_selected=0, n_links=0, n_chains=0, par_bit_exact=True, cov_bit_exact=True)
    gm = [tracker.get_tracks(s, B.OUT_MERGE | B.OUT_SELECTION).merge for s in range(tf.n_sectors)]
    for s in range(tf.n_sectors):
        g = gm[s]
        m = mg[s]
        rep = {}
        try:
            if g is None:
                raise ParityError("no S8 outputs delivered")
            for f in ("next_sec", "next_trk", "prev_sec", "prev_trk"):
                _eq("mg_" + f, g[f], getattr(m, f), rep)
            nk = len(m.next_sec)
            n_seg = np.zeros(nk, np.int32); n_seg[m.head] = m.n_seg
            _eq("mg_n_seg", g["n_seg"], n_seg, rep)
            h = m.head
            for f in ("n_hits", "n_fit", "first_row", "last_row", "frame_seg"):
                _eq("mg_" + f, g[f][h], getattr(m, f), rep)
            _eq("mg_x_ref", g["x_ref"][h], m.x_ref.astype(np.float32), rep)
            _eq("mg_z_ref", g["z_ref"][h], m.z_ref.astype(np.float32), rep)
            # the chain of every head, walked along the TRACKER's next links (gm, never the oracle's mg), equals the
            # oracle's segment list
            for k, ih in enumerate(h):
                segs = [(s, int(ih))]
                while len(segs) <= 4 * tf.n_sectors:          # a cycle in the GPU's links would fail the comparison below
                    a, b = segs[-1]
                    ga = gm[a]
                    if ga is None:
                        raise ParityError(f"chain of head {ih} enters sector {a}, which delivered no S8 outputs")
                    if ga["next_sec"][b] < 0:
                        break
                    segs.append((int(ga["next_sec"][b]), int(ga["next_trk"][b])))
                want = list(zip(m.seg_sec[m.seg_offset[k]:m.seg_offset[k + 1]].tolist(), m.seg_trk[m.seg_offset[k]:m.seg_offset[k + 1]].tolist()))
                if segs != want:
                    raise ParityError(f"chain of head {ih}: {segs} vs {want}")
            if len(h):
                gp = g["par"][h].astype(np.float64); op = m.par
                tol = 1e-4 * np.maximum(np.maximum(np.abs(gp), np.abs(op)), PAR_FLOOR[None, :])
                if (np.abs(gp - op) > tol).any():
                    t, i = np.argwhere(np.abs(gp - op) > tol)[0]
                    raise ParityError(f"mg_par[{t},{i}]: gpu {gp[t, i]} oracle {op[t, i]}")
                gc = g["cov"][h].astype(np.float64); oc = m.cov
                diag = np.stack([oc[:, i * (i + 1) // 2 + i] for i in range(5)], axis=1)
                for kk, (i, j) in enumerate(TRI):
                    lim = 1e-4 * np.sqrt(np.abs(diag[:, i] * diag[:, j]))
                    if (np.abs(gc[:, kk] - oc[:, kk]) > lim).any():
                        raise ParityError(f"mg_cov[{kk}] differs")
                g2 = g["chi2"][h].astype(np.float64)
                if (np.abs(g2 - m.chi2) > 1e-4 * np.maximum(np.maximum(np.abs(g2), np.abs(m.chi2)), 1e-3)).any():
                    raise ParityError("mg_chi2 differs")
                tot["par_bit_exact"] &= bool(np.array_equal(g["par"][h], op.astype(np.float32)))
                tot["cov_bit_exact"] &= bool(np.array_equal(g["cov"][h], oc.astype(np.float32)))
        except ParityError as e:
            raise ParityError(f"sector {s}: {e}") from None
        tot["sectors"] += 1; tot["n_selected"] += nk; tot["n_links"] += int((m.next_sec >= 0).sum()); tot["n_chains"] += len(h)
    return tot
