"""Randomized parity stress (not collected by pytest; run by hand on a B200: python tests/stress_parity.py [seconds]).

Seeded time frames of four recipes, a new seed each, through the CUDA path (S1-S8, every other one on a 0xff-poisoned
workspace) and the oracle: S1-S5 of 8 sectors, S6 of 3, S7 of 2, S8 of all 36, element by element.  Last run:
profiles/r2_stress.md."""
import sys, os, time
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT); sys.path.insert(0, os.path.join(ROOT, "tests"))
import numpy as np, tpcsynth
import paper_2208_07412_b200 as pkg
from oracle import Oracle
from parity import compare_timeframe, compare_selection, compare_residuals, compare_merge
t0=time.time(); n=0
budget=float(sys.argv[1]) if len(sys.argv)>1 else 600
seed=1000
while time.time()-t0 < budget:
    for cfg,kw in ((1,dict(n_tracks=2500)),(4,dict(n_tracks=1800)),(2,dict(n_orbits=1,mult_scale=0.6)),(2,dict(n_orbits=1,mult_scale=2.75))):
        seed+=1
        tf=tpcsynth.generate(cfg, seed=seed, **kw)
        trk=pkg.Tracker(tf.params, max_clusters=tf.n_clusters, workspace_fill=0xff if seed%2 else None)
        trk.load_timeframe(tf); trk.run(0xFF); trk.sync()
        orc=Oracle(tf.params)
        secs=list(range(0,36,5))
        try:
            r=compare_timeframe(trk, tf, orc, sectors=secs)
            compare_selection(trk, tf, orc, sectors=secs[:3])
            compare_residuals(trk, tf, orc, sectors=secs[3:5])
            m=compare_merge(trk, tf)
            print(f"seed {seed} cfg {cfg} {kw} n={tf.n_clusters} tracks={r['n_tracks']} links={m['n_links']} chains={m['n_chains']} par_exact={r['par_bit_exact']} mg_exact={m['par_bit_exact']} ok", flush=True)
        except AssertionError as e:
            print(f"seed {seed} cfg {cfg} {kw} FAIL: {e}", flush=True)
        trk.close(); n+=1
print("done", n, "cases in", time.time()-t0)
