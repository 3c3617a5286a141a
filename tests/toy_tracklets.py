"""Reader of tests/golden/toy_tracklets.txt (the hand-worked S5 decision toy) and the comparison of a
result (oracle or CUDA path: anything with order / hit_offset / hit_idx / first_row / last_row /
n_hits / n_fit / x_ref) against its hand-written expectations.  Holds none of the tracker's arithmetic."""
from __future__ import annotations

import os

import numpy as np

import tpcsynth

PATH = os.path.join(os.path.dirname(__file__), "golden", "toy_tracklets.txt")
N_ROWS = 32
SIGMA = 0.125


def _rows(spec):
    out = []
    if spec == "none":
        return out
    for part in spec.split(","):
        a, _, b = part.partition("-")
        out.extend(range(int(a), int(b or a) + 1))
    return out


class Scenario:
    def __init__(self, name, overrides):
        self.name = name
        self.overrides = overrides
        self.row, self.y, self.z = [], [], []
        self.tracks = {}          # name -> dict(y, z, expect: {row: cluster id}, emitted: bool)
        self.ties = []            # (win id, lose id, track name)

    def params(self):
        P = tpcsynth.default_params(n_sectors=1, row_x=64.0 + np.arange(N_ROWS), sigma=SIGMA)
        for k, v in self.overrides.items():
            assert hasattr(P, k), k
            setattr(P, k, type(getattr(P, k))(v))
        return P

    def arrays(self, reverse_ids=False):
        """(y, z, row) in original-id order; with reverse_ids cluster i becomes n-1-i."""
        y = np.array(self.y, np.float32); z = np.array(self.z, np.float32); row = np.array(self.row, np.uint16)
        assert np.array_equal(y.astype(np.float64), np.array(self.y)) and np.array_equal(z.astype(np.float64), np.array(self.z))
        if reverse_ids:
            return y[::-1].copy(), z[::-1].copy(), row[::-1].copy()
        return y, z, row

    def expected(self, reverse_ids=False):
        """{track name: sorted list of (file-order) cluster ids} of the tracks that must be emitted."""
        exp = {}
        swap = {}
        if reverse_ids:
            for w, l, _ in self.ties:
                swap[w] = l
        for name, t in self.tracks.items():
            if t["emitted"]:
                exp[name] = sorted(swap.get(c, c) for c in t["members"])
        return exp


def load():
    scen, cur = [], None
    last_tie = {}
    for line in open(PATH):
        line = line.split("#")[0].strip()
        if not line:
            continue
        f = line.split()
        kv = dict(p.split("=", 1) for p in f[2:])
        if f[0] == "scenario":
            cur = Scenario(f[1], {k: float(v) for k, v in kv.items()})
            scen.append(cur)
        elif f[0] == "track":
            y0, z0 = float(kv["y"]), float(kv["z"])
            exp_rows = set(_rows(kv["expect"]))
            members = []
            for r in _rows(kv["rows"]):
                cid = len(cur.row)
                cur.row.append(r); cur.y.append(y0); cur.z.append(z0)
                if r in exp_rows:
                    members.append(cid)
            assert exp_rows <= set(_rows(kv["rows"]))
            cur.tracks[f[1]] = dict(y=y0, z=z0, members=members, emitted=kv["expect"] != "none")
        elif f[0] == "extra":
            t = cur.tracks[f[1]]
            cid = len(cur.row)
            cur.row.append(int(kv["row"])); cur.y.append(t["y"] + float(kv["dy"])); cur.z.append(t["z"] + float(kv["dz"]))
            e = kv["expect"]
            assert e in ("in", "out", "tie-win", "tie-lose")
            if e in ("in", "tie-win"):
                t["members"].append(cid)
            if e == "tie-win":
                last_tie[f[1]] = cid
            if e == "tie-lose":
                cur.ties.append((last_tie.pop(f[1]), cid, f[1]))
        else:
            raise ValueError(line)
    assert not last_tie
    return scen


def check_result(sc: Scenario, res, reverse_ids=False):
    """Assert that `res` (one sector) holds exactly the expected tracks with the expected members."""
    n = len(sc.row)
    exp = sc.expected(reverse_ids)
    to_file_id = (lambda a: n - 1 - a) if reverse_ids else (lambda a: a)
    got = {}
    rows = np.array(sc.row)
    for t in range(res.n_tracks):
        hits = res.hit_idx[res.hit_offset[t]:res.hit_offset[t + 1]]
        ids = sorted(int(to_file_id(int(res.order[h]))) for h in hits)
        got[tuple(ids)] = t
    want = {tuple(v): k for k, v in exp.items()}
    missing = [want[k] for k in want if k not in got]
    extra = [k for k in got if k not in want]
    assert not missing and not extra, f"scenario {sc.name}: tracks not found as expected {missing}; unexpected tracks {extra}"
    assert res.n_tracks == len(exp)
    for ids, t in got.items():
        r = rows[list(ids)]
        assert res.first_row[t] == r.min() and res.last_row[t] == r.max() and res.n_hits[t] == len(ids)
        # reading N13: reference plane = lowest updated row; every hit above it was refitted
        assert res.n_fit[t] == len(ids) and float(res.x_ref[t]) == 64.0 + r.min(), want[ids]
