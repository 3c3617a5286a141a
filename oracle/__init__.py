"""CPU oracle of the TPC sector CA tracker -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` leg
may import this package.  It never imports the product package and the product never
imports it.
"""
from .binding import Oracle, OracleResult, MergeResult, run_timeframe, run_timeframe_merged, select_tracks, merge_links_of_tables

__all__ = ["Oracle", "OracleResult", "run_timeframe", "run_timeframe_merged", "select_tracks", "merge_links_of_tables", "MergeResult"]
