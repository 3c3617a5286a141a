"""Seeded synthetic ALICE-TPC-shaped inputs and the tracker's data tables.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the tracker's arithmetic (no binning, no link scores, no Kalman filter):
only (a) the geometry / window / cut tables, which are *data* handed verbatim to
both implementations, and (b) the seeded generators of BASELINE.json configs
0-4 together with their generator-truth bookkeeping.
"""
from .params import TrackerParams, default_params, BC_PER_QPT, V_DRIFT, ORBIT_US
from .generator import (CONFIGS, Timeframe, generate,
                        truth_state, straight_tracks, helix_hits)

__all__ = ["TrackerParams", "default_params", "BC_PER_QPT", "V_DRIFT", "ORBIT_US",
           "CONFIGS", "Timeframe", "generate", "truth_state",
           "straight_tracks", "helix_hits"]
