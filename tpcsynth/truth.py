"""Generator-truth bookkeeping: efficiency / clone / fake rates of a set of found tracks.

Definitions (SURVEY.md section 8(c) pin P10): a generated track is *findable in a sector* if it
left >= 20 clusters there; a found track *matches* a generated track if >= 90 % of its hits
carry that track's label; efficiency = findable (track, sector) pairs with >= 1 match /
findable pairs; clone rate = (matches - matched pairs) / matches; fake rate = found tracks
matching nothing / found tracks.  Pure bookkeeping on labels: none of the tracker's
arithmetic lives here.
"""
from __future__ import annotations

import numpy as np


def match_tracks(label_sorted: np.ndarray, hit_offset: np.ndarray, hit_idx: np.ndarray, purity: float = 0.9):
    """Per found track: (majority label or -1 if below purity, purity)."""
    n_trk = hit_offset.shape[0] - 1
    maj = np.full(n_trk, -1, dtype=np.int64)
    pur = np.zeros(n_trk)
    for t in range(n_trk):
        labs = label_sorted[hit_idx[hit_offset[t]:hit_offset[t + 1]]]
        labs = labs[labs >= 0]
        n = hit_offset[t + 1] - hit_offset[t]
        if labs.size == 0 or n == 0:
            continue
        vals, cnt = np.unique(labs, return_counts=True)
        k = int(np.argmax(cnt))
        pur[t] = cnt[k] / n
        if pur[t] >= purity:
            maj[t] = vals[k]
    return maj, pur


def sector_metrics(label: np.ndarray, order: np.ndarray, hit_offset: np.ndarray, hit_idx: np.ndarray,
                   min_findable: int = 20, purity: float = 0.9) -> dict:
    """Efficiency / clone / fake counts for one sector.

    label: per original cluster; order: sorted -> original; hit_idx: sorted positions.
    """
    label_sorted = label[order]
    maj, _ = match_tracks(label_sorted, hit_offset, hit_idx, purity)
    sig = label[label >= 0]
    ids, cnt = np.unique(sig, return_counts=True)
    findable = set(ids[cnt >= min_findable].tolist())
    matched = maj[maj >= 0]
    found_ids = set(matched.tolist())
    n_found_findable = len(findable & found_ids)
    return dict(n_findable=len(findable), n_found=n_found_findable,
                n_tracks=int(maj.shape[0]), n_matched=int(matched.shape[0]),
                n_fake=int((maj < 0).sum()), n_distinct_matched=len(found_ids))


def summarize(ms) -> dict:
    tot = {k: sum(m[k] for m in ms) for k in ms[0]}
    tot["efficiency"] = tot["n_found"] / max(tot["n_findable"], 1)
    tot["fake_rate"] = tot["n_fake"] / max(tot["n_tracks"], 1)
    tot["clone_rate"] = (tot["n_matched"] - tot["n_distinct_matched"]) / max(tot["n_matched"], 1)
    return tot
