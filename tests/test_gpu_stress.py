"""Randomized parity stress of the CUDA path against the oracle, S1-S8.

Seeded time frames of four recipes (config-1 and config-4 kinematics, one orbit of the time-frame config at low and
at 2.75x occupancy), a new seed each, every other one on a 0xff-poisoned workspace: S1-S5 of 8 sectors, S6 of 3, S7 of
2 and S8 of all 36, element by element.  By default ONE pass over the four recipes (seconds); the long run of
profiles/r2_stress.md is `TPCCA_STRESS_SECONDS=1200 python -m pytest tests/test_gpu_stress.py -m gpu -s`.
"""
import os
import time

import pytest

import tpcsynth
from oracle import Oracle
from parity import compare_merge, compare_residuals, compare_selection, compare_timeframe

pytestmark = pytest.mark.gpu

RECIPES = ((1, dict(n_tracks=2500)), (4, dict(n_tracks=1800)), (2, dict(n_orbits=1, mult_scale=0.6)),
           (2, dict(n_orbits=1, mult_scale=2.75)))


def test_seeded_time_frames_s1_to_s8():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    import paper_2208_07412_b200 as pkg
    budget = float(os.environ.get("TPCCA_STRESS_SECONDS", "0"))
    t0, seed, n_cases, n_clusters = time.time(), 3000, 0, 0
    while True:
        for cfg, kw in RECIPES:
            seed += 1
            tf = tpcsynth.generate(cfg, seed=seed, **kw)
            trk = pkg.Tracker(tf.params, max_clusters=tf.n_clusters, workspace_fill=0xff if seed % 2 else None)
            trk.load_timeframe(tf)
            trk.run(0xFF)
            trk.sync()
            orc = Oracle(tf.params)
            secs = list(range(0, 36, 5))
            r = compare_timeframe(trk, tf, orc, sectors=secs)
            compare_selection(trk, tf, orc, sectors=secs[:3])
            compare_residuals(trk, tf, orc, sectors=secs[3:5])
            m = compare_merge(trk, tf)
            trk.close()
            assert r["links_differing"] == 0, (seed, cfg, kw, r)      # (a Poisson draw of zero collisions gives an empty time frame)
            assert tf.n_clusters < 100000 or (r["n_tracks"] > 0 and m["n_links"] > 0), (seed, cfg, kw, r, m)
            print(f"seed {seed} cfg {cfg} {kw} n={tf.n_clusters} tracks={r['n_tracks']} links={m['n_links']} "
                  f"chains={m['n_chains']} par_exact={r['par_bit_exact']} mg_exact={m['par_bit_exact']} ok", flush=True)
            n_cases += 1; n_clusters += tf.n_clusters
        if time.time() - t0 >= budget:
            break
    print(f"{n_cases} time frames, {n_clusters} clusters in {time.time() - t0:.0f} s")
