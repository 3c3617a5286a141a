#!/usr/bin/env python
"""bench.py -- throughput of the TPC sector CA tracker hot path (S1-S5) on B200.

Contract: `python bench.py --gpus N --steps K --warmup W [--impl reference]` prints ONE JSON line.
A step = one pass of the whole hot path (tpcca_run(S1..S5)) over one synthetic time frame.
Workload at N=1: BASELINE.json configs[3] (128-orbit 50 kHz Pb-Pb-like time frame, seeded synthetic,
tpcsynth recipe of DESIGN.md 6).  N>1: one time frame per GPU (the paper's own scheme, PAPER.md:21
"different collisions are distributed over the EPNs"): replicas, no data-path collective, weak scaling.

  value     : clusters/s, inputs resident in HBM before the timed region (device-timed, max over ranks)
  e2e       : same metric through the C-ABI with HOST (pinned) buffers: H2D of the clusters and D2H of
              order + cleaned links + start hits + track table + hit CSR inside the timed region
  roofline  : neighbour finder (S2; the stage BASELINE.json's metric names) vs the measured HBM peak;
  roofline_dominant : the stage that takes the most time (S5 tracklets), plain-ALU bound
  cpu_baseline : the oracle as it stands, one single-threaded oracle per sector job over all host cores, on all 36
                 sectors of the same time frame (wall clock); 8 sectors spread over both sides are then compared
                 element by element with the CUDA path (the full-size parity check)
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np

METRIC = "TPC clusters tracked/sec per B200 (full timeframe)"
UNIT = "clusters/s"

# fp32 operations of one call, counted from DESIGN.md 3.5 (every + - * / sqrt is one operation)
FLOPS_PROPAGATE = 157   # 55 transport + 52 (A = J C) + 50 (C' = A J^T)
FLOPS_UPDATE = 102      # 2 x (1 + 2 + 5 + 10 + 30 + 3)
FLOPS_GATE = 9
FLOPS_SEARCH = 23       # bin range + weights
FLOPS_CANDIDATE = 10


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback (B200_PROFILING.md: 6.65 TB/s)")


def ncu_traffic(args, n_clusters):
    """dram bytes read + written per launch of the S2 kernels from the committed ncu capture of this workload
    (profiles/r2_traffic.txt), or None when the workload differs from the captured one."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.txt")
    if not os.path.exists(p):
        return None
    d = json.load(open(p))
    if d.get("config") != args.config or d.get("n_clusters") != n_clusters:
        return None
    return float(d["s2_dram_bytes_per_launch"])


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for t, line in self.lines:
            if t < t0 - 0.05 or t > t1 + 0.15:
                continue
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))


def rank_seed(config, seed, rank):
    """Seed of the time frame rank `rank` tracks: the config's default seed on rank 0 (so the N = 1 workload is
    exactly BASELINE.json's), a distinct one on every other rank (replicas process DIFFERENT time frames)."""
    import tpcsynth
    base = seed if seed is not None else tpcsynth.generator.BASE_SEED + config
    return base + 1000 * rank


def reduce_over_ranks(v, op, world, dev):
    """max / sum of a host scalar over the ranks (identity for world == 1); NCCL on GPU, gloo in the CPU tests."""
    if world == 1:
        return v
    import torch
    import torch.distributed as dist
    t = torch.tensor([v], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_value(n_local, steps, ms_local, world, dev):
    """Whole-job throughput: units all ranks processed / the slowest rank's device time."""
    ms = reduce_over_ranks(ms_local, "max", world, dev)
    n_all = reduce_over_ranks(float(n_local), "sum", world, dev)
    return n_all * steps / (ms * 1e-3), ms, n_all


def make_timeframe(args, rank):
    import tpcsynth
    t0 = time.time()
    tf = tpcsynth.generate(args.config, seed=rank_seed(args.config, args.seed, rank), mult_scale=args.mult_scale)
    return tf, time.time() - t0


def sample_sector(tf, sector, z_frac):
    """Bounded sample of the workload: clusters of one sector with z below z_frac of the z range."""
    y, z, row = tf.y[sector], tf.z[sector], tf.row[sector]
    if z_frac >= 1.0:
        return y, z, row
    m = z < np.float32(z_frac * tf.params.z_hi)
    return np.ascontiguousarray(y[m]), np.ascontiguousarray(z[m]), np.ascontiguousarray(row[m])


def workload_name(args, tf):
    import tpcsynth
    return (f"BASELINE.json configs[{args.config}] ({tpcsynth.CONFIGS[args.config]['name']}), seed {tf.seed}, "
            f"mult_scale {args.mult_scale}")


# --------------------------------------------------------------------------------------------------
def run_reference(args):
    """The oracle (CPU, one core) on bounded samples of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import Oracle
    tf, gen_s = make_timeframe(args, 0)
    y, z, row = sample_sector(tf, 0, args.ref_z_frac)
    orc = Oracle(tf.params)
    for _ in range(args.warmup):
        orc.run(y, z, row, want=())
    t0 = time.time()
    for _ in range(args.steps):
        orc.run(y, z, row, want=())
    dt = time.time() - t0
    n = int(y.shape[0])
    value = n * args.steps / dt
    sample = f"sector 0 of {tf.n_sectors}, z < {args.ref_z_frac:g} of the z range: {n} of {tf.n_clusters} clusters per step"
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=1e3 * dt / args.steps, higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f32", data="synthetic",
                config=dict(workload=workload_name(args, tf), n_clusters=tf.n_clusters, sample=sample),
                cpu_baseline=dict(value=value, unit=UNIT, cores=1, kind="oracle", sample=sample),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                gpu_launches=0, generate_s=gen_s)
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------
def _oracle_timed_job(job):
    """Worker of the CPU-baseline pool (a spawned process: no CUDA in here): the oracle as it stands on one
    sector, S1-S5 (the five stages of the hot path) without output copies; returns the seconds it took."""
    params, y, z, row = job
    from oracle import Oracle
    orc = Oracle(params)
    t0 = time.time()
    orc.run(y, z, row, want=())
    return time.time() - t0


def _oracle_output_job(job):
    """Worker: the full OracleResult of one sector, S6 / S7 included, for the parity check (not timed)."""
    params, y, z, row = job[:4]
    from oracle import Oracle
    return Oracle(params).run(y, z, row, stage_mask=job[4] if len(job) > 4 else 0x7F)


def merge_properties(trk, tf, B):
    """S8 at full size, where the oracle's all-pairs matching is out of reach: properties that hold at any size.  Links are
    mutual, join neighbouring sectors of one side, the upper segment starts 1 .. mg_max_row_gap rows above the lower one,
    and every chain head's segment count equals the length of its link chain."""
    P = tf.params
    per, ns = P.sectors_per_side, tf.n_sectors
    outs = [trk.get_tracks(s, B.OUT_MERGE | B.OUT_TRACKS_SEL) for s in range(ns)]
    n_links = n_chains = n_fitted = 0
    for s, o in enumerate(outs):
        m = o.merge
        a = np.nonzero(m["next_sec"] >= 0)[0]
        if a.size == 0:
            continue
        nsec, ntrk = m["next_sec"][a], m["next_trk"][a]
        assert np.all(nsec // per == s // per) and np.all(np.isin((nsec % per - s % per) % per, (1, per - 1))), "not neighbours"
        for t in np.unique(nsec):
            sel = nsec == t
            b = outs[t]
            assert np.array_equal(b.merge["prev_sec"][ntrk[sel]], np.full(sel.sum(), s)), "prev_sec not mutual"
            assert np.array_equal(b.merge["prev_trk"][ntrk[sel]], a[sel]), "prev_trk not mutual"
            gap = b.first_row[ntrk[sel]] - o.last_row[a[sel]]
            assert gap.min() >= 1 and gap.max() <= P.mg_max_row_gap, "row gap out of range"
        n_links += int(a.size)
        heads = np.nonzero((m["prev_sec"] < 0) & (m["next_sec"] >= 0))[0]
        fitted = np.nonzero(m["n_seg"] > 0)[0]                  # (a chain whose top segment has no outer state is not refitted)
        assert np.all(np.isin(fitted, heads)), "chain heads"
        n_fitted += int(fitted.size)
        for h in fitted[:: max(1, fitted.size // 200)]:        # a sample of the chains is walked
            k, cs, ct = 1, s, int(h)
            while outs[cs].merge["next_sec"][ct] >= 0:
                cs, ct = int(outs[cs].merge["next_sec"][ct]), int(outs[cs].merge["next_trk"][ct])
                k += 1
            assert k == m["n_seg"][h], "n_seg"
        n_chains += int(heads.size)
    return dict(status="pass", n_links=n_links, n_chains=n_chains, n_refitted=n_fitted)


def cpu_baseline_and_parity(args, tf, trk):
    """CPU baseline: the oracle as it stands on `--cpu-sectors` sectors (default: all of them),
    one single-threaded oracle per sector job spread over ALL host cores of the box, wall clock around the pool.
    Then the oracle's full outputs of `--parity-sectors` sectors spread over both sides are computed (not timed) and
    compared element by element with the CUDA path's outputs of the same sectors."""
    import multiprocessing as mp
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from oracle import Oracle
    from parity import compare_sector
    ns = tf.n_sectors
    spread = lambda k: sorted({(i * ns) // k for i in range(max(1, min(k, ns)))})
    timed, sectors = spread(args.cpu_sectors), spread(args.parity_sectors)
    avail = len(os.sched_getaffinity(0))
    cores = min(len(timed), avail)
    job = lambda s: (tf.params, tf.y[s], tf.z[s], tf.row[s])
    # largest sectors first, so that the last wave is not one long job on an otherwise idle pool
    timed_jobs = [job(s) for s in sorted(timed, key=lambda s: -tf.y[s].shape[0])]
    with mp.get_context("spawn").Pool(cores) as pool:
        pool.map(int, range(4 * cores))                  # workers up (interpreter + numpy imported) before the clock starts
        t0 = time.time()
        dts = pool.map(_oracle_timed_job, timed_jobs, chunksize=1)
        wall = time.time() - t0
        out = pool.map(_oracle_output_job, [job(s) for s in sectors], chunksize=1)
    n_s = int(sum(tf.y[s].shape[0] for s in timed))
    busy = float(sum(dts))
    cpu = dict(value=float(n_s / wall), unit=UNIT, cores=cores, kind="oracle",
               sample=f"{len(timed)} of {ns} sectors: {n_s} of {tf.n_clusters} clusters, S1-S5, one single-threaded oracle per "
                      f"sector over {cores} of the box's {avail} host cores: {wall:.1f} s wall ({busy:.1f} core-s)",
               one_core_value=float(n_s / busy))
    orc = Oracle(tf.params)
    parity = dict(sectors=sectors, n_clusters=0, n_tracks=0, links_differing=0, membership="bit-exact",
                  par_bit_exact=True, n_selected=0, n_attached=0, s6_s7="bit-exact", status="pass")
    B = sys.modules["paper_2208_07412_b200.binding"]
    trk.run(0xFF)                                    # the same time frame once more, S6 - S8 included
    trk.sync()
    try:
        parity["s8_properties"] = merge_properties(trk, tf, B)
    except AssertionError as e:
        parity.update(status="FAIL", error=f"S8 properties: {str(e)[:300]}")
    for s, o in zip(sectors, out):
        g = trk.get_tracks(s, B.OUT_ALL | B.OUT_SELECTION | B.OUT_RESIDUALS)
        try:
            rep = compare_sector(g, o, orc, tf.row[s][o.order])
            for f in ("owner", "n_own", "selected", "res_trk", "q_y", "q_z"):
                if not np.array_equal(getattr(g, f), getattr(o, f)):
                    raise AssertionError(f"S6/S7 output {f} differs")
            for f in ("res_y", "res_z"):
                if not np.array_equal(getattr(g, f), getattr(o, f).astype(np.float32)):
                    raise AssertionError(f"S7 output {f} differs")
            parity["n_selected"] += int(len(o.selected)); parity["n_attached"] += int((o.res_trk >= 0).sum())
        except AssertionError as e:
            parity.update(status="FAIL", error=f"sector {s}: {str(e)[:300]}")
            break
        parity["n_clusters"] += int(o.n); parity["n_tracks"] += int(o.n_tracks)
        parity["links_differing"] += rep["links_differing"]
        parity["par_bit_exact"] = bool(parity["par_bit_exact"] and rep.get("par_bit_exact", True))
    return cpu, parity


def footprint_leg(args, env, peaks):
    """The footprint BASELINE.json:10 names for the headline workload ("about 4e8 clusters (~8 GB fp32 SoA)"): the
    generator text of configs[3] yields 1.45e8 clusters ("discrepancy to carry forward"), so the
    same recipe is run once more at mult_scale 2.75 (~4e8 clusters): W warm-ups + 3 timed steps of S1-S5 on
    device-resident inputs, per-stage times, the S2 roofline fraction, and an element-by-element parity check of two
    sectors (one per side) against the oracle.  Called after the main legs have released their contexts."""
    import copy
    import multiprocessing as mp
    import tpcsynth
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from oracle import Oracle
    from parity import compare_sector
    B = env.B
    a = copy.copy(args)
    a.mult_scale = args.footprint_scale
    t0 = time.time()
    tf = tpcsynth.generate(a.config, seed=rank_seed(a.config, a.seed, 0), mult_scale=a.mult_scale)
    gen_s = time.time() - t0
    N = tf.n_clusters
    sectors = [0, tf.n_sectors // 2] if tf.n_sectors > 1 else [0]
    pool = mp.get_context("spawn").Pool(len(sectors))       # the oracle starts on its sectors while the GPU leg runs
    orc_async = pool.map_async(_oracle_output_job, [(tf.params, tf.y[s], tf.z[s], tf.row[s], 0x1F) for s in sectors], chunksize=1)
    trk = env.tracker(tf.params, N, N // 8 + 1024)
    devin = [(env.to_device(env.pin(tf.y[s])), env.to_device(env.pin(tf.z[s])), env.to_device(env.pin_u16(tf.row[s])))
             for s in range(tf.n_sectors)]
    trk.reset()
    for s, (y, z, r) in enumerate(devin):
        trk.load_clusters(s, y, z, r, borrow=True)
    for _ in range(args.warmup):
        trk.run()
    trk.sync()
    steps = 3
    ev0, ev1 = env.event(), env.event()
    env.synchronize()
    ev0.record()
    for _ in range(steps):
        trk.run()
    ev1.record()
    env.synchronize()
    ms = ev0.elapsed_time(ev1) / steps
    trk.sync()
    stage_ms = np.mean([trk.timings(i) for i in range(steps)], axis=0)
    counts = trk.counts()
    s2_bytes = 16.0 * N + 4.0 * counts["n_bins"] * tf.n_sectors
    s2_gbs = s2_bytes / (stage_ms[1] * 1e-3) / 1e9
    res = dict(workload=workload_name(a, tf), n_clusters=N, soa_bytes=int(18 * N), steps=steps, warmup=args.warmup,
               ms_per_step=ms, value=N / (ms * 1e-3), unit=UNIT, n_start=counts["n_start"], n_tracks=counts["n_tracks"],
               stage_ms=dict(zip(("S1_grid", "S2_neighbours", "S3_clean", "S4_start", "S5_tracklets", "total"),
                                 (round(float(v), 4) for v in stage_ms))),
               roofline=dict(kernel="S2 neighbour finder", bound="hbm", achieved=s2_gbs, peak=peaks["hbm_gbs"], unit="GB/s",
                             frac=s2_gbs / peaks["hbm_gbs"], algorithmic_bytes=s2_bytes),
               generate_s=round(gen_s, 1))
    parity = dict(sectors=sectors, n_clusters=0, n_tracks=0, links_differing=0, par_bit_exact=True, status="pass")
    t0 = time.time()
    outs = orc_async.get()
    pool.close()
    parity["oracle_wait_s"] = round(time.time() - t0, 1)
    orc = Oracle(tf.params)
    for s, o in zip(sectors, outs):
        g = trk.get_tracks(s, B.OUT_ALL)
        try:
            rep = compare_sector(g, o, orc, tf.row[s][o.order])
        except AssertionError as e:
            parity.update(status="FAIL", error=f"sector {s}: {str(e)[:300]}")
            break
        parity["n_clusters"] += int(o.n); parity["n_tracks"] += int(o.n_tracks)
        parity["links_differing"] += rep["links_differing"]
        parity["par_bit_exact"] = bool(parity["par_bit_exact"] and rep.get("par_bit_exact", True))
    res["parity"] = parity
    trk.close()
    devin.clear()
    env.empty_cache()
    return res


# --------------------------------------------------------------------------------------------------
class CudaEnv:
    """Everything run_tpcca needs from the device side: the tpcca Tracker (the product), torch.cuda for device
    memory / streams / events, NCCL for the barrier and the reductions.  tests/test_multirank.py swaps it for a
    CPU stand-in (gloo, a stub Tracker) to drive the N > 1 host logic of run_tpcca without a GPU."""
    backend = "nccl"

    def __init__(self, rank, world, local):
        import torch
        import paper_2208_07412_b200 as pkg
        from paper_2208_07412_b200 import binding as B
        if not torch.cuda.is_available():
            raise RuntimeError(f"bench.py rank {rank}/{world}: needs a CUDA device: tpcca has no CPU path")
        torch.cuda.set_device(local)
        self.torch, self.pkg, self.B = torch, pkg, B
        self.local = local
        self.device = torch.device(f"cuda:{local}")
        self.oom_error = torch.OutOfMemoryError

    def init_process_group(self):
        import torch.distributed as dist
        dist.init_process_group(self.backend, device_id=self.device)

    def tracker(self, params, max_clusters, max_start_hits, stream=None):
        return self.pkg.Tracker(params, max_clusters=max_clusters, max_start_hits=max_start_hits, device=self.local, stream=stream)

    def pipeline(self, params, n_groups, max_clusters_group, max_start_hits_group):
        return self.pkg.Pipeline(params, n_groups, max_clusters_group, max_start_hits_group, device=self.local)

    def pin(self, a):
        return self.torch.from_numpy(a).pin_memory()

    def pin_u16(self, a):
        return self.torch.from_numpy(a.view(np.int16)).pin_memory().view(self.torch.uint16)

    def to_device(self, t):
        return t.to(self.device)

    def event(self):
        return self.torch.cuda.Event(enable_timing=True)

    def synchronize(self):
        self.torch.cuda.synchronize()

    def set_thread_device(self):
        self.torch.cuda.set_device(self.local)       # a new host thread starts on device 0

    def stream(self):
        return self.torch.cuda.Stream(device=self.device)

    def wait_stream(self, sd):
        self.torch.cuda.current_stream().wait_stream(sd)

    def empty_cache(self):
        self.torch.cuda.empty_cache()

    def sm_count(self):
        return self.torch.cuda.get_device_properties(self.local).multi_processor_count

    def clock_sampler(self):
        return ClockSampler(self.local)


def run_tpcca(args, env_cls=CudaEnv):
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    env = env_cls(rank, world, local)
    B = env.B
    if world > 1:
        env.init_process_group()
    dev = env.device

    def barrier():
        if world > 1:
            dist.barrier()
        env.synchronize()

    def max_over_ranks(v):
        return reduce_over_ranks(v, "max", world, dev)

    def sum_over_ranks(v):
        return reduce_over_ranks(v, "sum", world, dev)

    peaks = load_peaks()
    tf, gen_s = make_timeframe(args, rank)
    N = tf.n_clusters
    cap = args.max_start_hits or (N // 8 + 1024)
    trk = env.tracker(tf.params, N, cap)

    # ---- device-resident inputs (borrowed: no copy inside the timed region) ------------------------
    host = []
    for s in range(tf.n_sectors):
        host.append((env.pin(tf.y[s]), env.pin(tf.z[s]), env.pin_u16(tf.row[s])))
    devin = [(env.to_device(a), env.to_device(b), env.to_device(c)) for a, b, c in host]
    trk.reset()
    for s, (a, b, c) in enumerate(devin):
        trk.load_clusters(s, a, b, c, borrow=True)

    for _ in range(args.warmup):
        trk.run()
    trk.sync()
    launches_per_step = trk.launch_count()
    counts = trk.counts()

    sampler = env.clock_sampler()
    sampler.start()
    time.sleep(0.3)
    ev0, ev1 = env.event(), env.event()
    barrier()
    t_wall0 = time.time()
    ev0.record()
    for _ in range(args.steps):
        trk.run()
    ev1.record()
    env.synchronize()
    t_wall1 = time.time()
    barrier()
    value, ms_total, n_all = whole_job_value(N, args.steps, ev0.elapsed_time(ev1), world, dev)
    clocks = sampler.stop(t_wall0, t_wall1)
    trk.sync()

    # per-stage device times of the timed steps (events recorded inside tpcca_run on the same stream)
    k = min(args.steps, 16)
    stage_ms = np.mean([trk.timings(i) for i in range(k)], axis=0)
    work = trk.work_counters()
    n_bins_total = counts["n_bins"] * tf.n_sectors
    s2_bytes = 16.0 * N + 4.0 * n_bins_total
    s2_gbs = s2_bytes / (stage_ms[1] * 1e-3) / 1e9
    flops = (work["propagations"] * FLOPS_PROPAGATE + work["updates"] * FLOPS_UPDATE + work["gates"] * FLOPS_GATE
             + work["searches"] * FLOPS_SEARCH + work["candidates"] * FLOPS_CANDIDATE)
    n_sm = env.sm_count()
    alu_peak = n_sm * 128 * peaks["sm_max_mhz"] * 1e6 / 1e12      # T fp32 op/s without FMA
    s5_tops = flops / (stage_ms[4] * 1e-3) / 1e12

    # ---- end to end: host buffers in, host buffers out, through the public API ---------------------
    h2d = int(10 * N)

    def e2e_step(t, selected=False):
        """One whole step through the public API: pinned HOST inputs in, HOST outputs out.  selected: the step also
        runs S6 and ships the selected tracks (compact table) + per-cluster owner instead of every tracklet."""
        t.reset()
        for s, (a, b, c) in enumerate(host):
            t.load_clusters(s, a, b, c)
        t.run(0x3F if selected else 0x1F)
        out = 0
        early = B.OUT_ORDER | B.OUT_LINKS | B.OUT_START          # ready after S4: copied while S5 runs
        for s in range(tf.n_sectors):
            v = t.get_tracks_view(s, B.MEM_HOST, early)
            out += 12 * v.n_clusters + 4 * v.n_start
        for s in range(tf.n_sectors):
            if selected:
                v = t.get_tracks_view(s, B.MEM_HOST, B.OUT_TRACKS_SEL | B.OUT_SELECTION)
                out += 4 * v.n_sel_hits + (4 * 28 + 4) * v.n_selected + 4 + 4 * v.n_clusters + 4 * v.n_tracks + 4 * v.n_selected
            else:
                v = t.get_tracks_view(s, B.MEM_HOST, B.OUT_TRACKS)
                out += 4 * v.n_hits + (4 * 28 + 4) * v.n_tracks + 4
        return int(out)

    # (a) serial: one context, step after step
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    d2h = e2e_step(trk)   # warm-up: grows the pinned arena
    barrier()
    ev0.record()
    for _ in range(e2e_steps):
        e2e_step(trk)
    ev1.record()
    env.synchronize()
    barrier()
    e2e_serial_ms = max_over_ranks(ev0.elapsed_time(ev1))

    # (a') the same serial step with S6 on: the consumer downloads the selected tracks only
    d2h_sel = e2e_step(trk, True)
    barrier()
    ev0.record()
    for _ in range(e2e_steps):
        e2e_step(trk, True)
    ev1.record()
    env.synchronize()
    barrier()
    e2e_sel_serial_ms = max_over_ranks(ev0.elapsed_time(ev1))
    s6_ms = float(trk.timings(0)[6])
    counts_sel = trk.counts()
    # S7 residual front end and S8 cross-sector merging + chain refit on the same time frame (outside every timed
    # region): each stage twice, the faster run reported (the first launch of a kernel pays its module load)
    trk.run(0x40); s7_ms = float(trk.timings(0)[7])
    trk.run(0x40); s7_ms = min(s7_ms, float(trk.timings(0)[7]))
    trk.run(0x80); s8_ms = float(trk.timings(0)[8])
    trk.run(0x80); s8_ms = min(s8_ms, float(trk.timings(0)[8]))

    # (b) streaming (the EPN operating mode: time frames follow each other): two contexts on two
    # streams, each step still does its own H2D, S1-S5 and D2H, but the copies of one time frame overlap the
    # kernels of the other (PCIe is full duplex).  One host thread per context (ctypes releases the GIL).
    e2e_ms, e2e_n = e2e_serial_ms, e2e_steps
    e2e_mode = "serial, 1 context"
    e2e_sel_stream_ms = None
    if not args.no_streaming:
        n_ctx = max(2, args.e2e_contexts)
        sides = [env.stream() for _ in range(n_ctx - 1)]
        extra = []
        try:
            for sd in sides:
                extra.append(env.tracker(tf.params, N, cap, stream=sd))
        except env.oom_error:      # the workspace of another time frame does not fit beside the first
            for t in extra:
                t.close()
            extra = None
            env.empty_cache()
        if extra:
            per = e2e_steps

            def stream_leg(selected, serial_ms):
                for t in extra:
                    e2e_step(t, selected)          # warm-up: grows the pinned arenas
                env.synchronize()

                def worker(t, delay):
                    env.set_thread_device()
                    time.sleep(delay)              # the contexts start a fraction of a step apart: the copies of one meet the kernels of another
                    for _ in range(per):
                        e2e_step(t, selected)

                barrier()
                ev0.record()
                step_s = 1e-3 * serial_ms / e2e_steps
                th = [threading.Thread(target=worker, args=(t, i * step_s / n_ctx)) for i, t in enumerate([trk] + extra)]
                for t in th:
                    t.start()
                for t in th:
                    t.join()
                for sd in sides:
                    env.wait_stream(sd)
                ev1.record()
                env.synchronize()
                barrier()
                return max_over_ranks(ev0.elapsed_time(ev1))

            e2e_ms = stream_leg(False, e2e_serial_ms)
            e2e_n = n_ctx * per
            e2e_mode = "streaming, %d contexts on %d streams" % (n_ctx, n_ctx)
            e2e_sel_stream_ms = stream_leg(True, e2e_sel_serial_ms)
            for t in extra:
                t.close()
        else:
            e2e_mode = "serial, 1 context (no device memory for a second time frame)"
    # (c) one time frame through the sector-group pipeline of the library (tpcca_pipeline_run: SURVEY 8(f)-3): latency of
    # ONE time frame, host buffers in, host views out, the groups' copies overlapping each other's kernels
    pipe_res = None
    if args.pipeline_groups > 1 and world == 1:
        G = min(args.pipeline_groups, tf.n_sectors)
        first = [g * tf.n_sectors // G for g in range(G + 1)]
        sc = tf.sector_counts()
        cap_g = int(max(sc[first[g]:first[g + 1]].sum() for g in range(G)) * 1.05) + 1024
        try:
            pipe = env.pipeline(tf.params, G, cap_g, cap_g // 8 + 1024)
        except env.oom_error:
            pipe = None
        if pipe is not None:
            hy = [h[0] for h in host]; hz = [h[1] for h in host]; hr = [h[2] for h in host]

            def pipe_leg(mask, what, selected):
                pipe.run_views(hy, hz, hr, mask, what)          # warm-up: grows the pinned arenas
                env.synchronize()
                t0 = time.perf_counter()
                for _ in range(e2e_steps):
                    views = pipe.run_views(hy, hz, hr, mask, what)
                env.synchronize()
                dt = (time.perf_counter() - t0) / e2e_steps
                if selected:
                    nb = sum(12 * v.n_clusters + 4 * v.n_start + 4 * v.n_sel_hits + (4 * 28 + 4) * v.n_selected + 4
                             + 4 * v.n_clusters + 4 * v.n_tracks + 4 * v.n_selected for v in views)
                else:
                    nb = sum(12 * v.n_clusters + 4 * v.n_start + 4 * v.n_hits + (4 * 28 + 4) * v.n_tracks + 4 for v in views)
                gms = [round(v, 1) for v in pipe.groups()[1]]
                # the pipeline is a LATENCY mode: its figure of merit is when the first group's tracks
                # are on the host, not the throughput (two whole contexts, `e2e.value`, are faster per time frame)
                return dict(value=N / dt, unit=UNIT, ms_per_step=1e3 * dt, d2h_bytes_per_step=int(nb),
                            group_ms=gms, first_tracks_ms=min(gms))

            early = B.OUT_ORDER | B.OUT_LINKS | B.OUT_START
            pipe_res = pipe_leg(0x1F, early | B.OUT_TRACKS, False)
            pipe_res.update(n_groups=G, h2d_bytes_per_step=h2d,
                            mode=f"one time frame at a time, {G} sector groups on {G} streams / host threads (host wall clock)",
                            selected=pipe_leg(0x3F, early | B.OUT_TRACKS_SEL | B.OUT_SELECTION, True))
            pipe.close()
            env.empty_cache()
    e2e_value = n_all * e2e_n / (e2e_ms * 1e-3)
    e2e_steps_serial = e2e_steps
    e2e_steps = e2e_n

    # ---- CPU baseline = the oracle, one sector per host core, on a bounded sample of the sectors (rank 0,
    # N = 1 only); the same results are a full-size parity check of those sectors ----------------------------
    cpu = None
    parity = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu, parity = cpu_baseline_and_parity(args, tf, trk)

    # ---- the ~4e8-cluster footprint BASELINE.json:10 names, as a short extra leg (rank 0, N = 1, default workload) ----
    footprint = None
    if (rank == 0 and world == 1 and args.footprint_scale > 0 and args.config == 3 and args.mult_scale == 1.0
            and not args.no_cpu_baseline):
        trk.close()
        devin.clear(); host.clear()
        hy = hz = hr = None
        env.empty_cache()
        try:
            footprint = footprint_leg(args, env, peaks)
        except env.oom_error as e:
            footprint = dict(status="FAIL", error=f"out of memory: {str(e)[:200]}")

    if rank == 0:
        line = dict(
            metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
            ms_per_step=ms_total / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None,
            dtype="f32", data="synthetic",
            config=dict(workload=workload_name(args, tf), n_clusters_per_gpu=N, n_sectors=tf.n_sectors,
                        n_start=counts["n_start"], n_tracks=counts["n_tracks"], n_hits=counts["n_hits"],
                        grid_bins=n_bins_total, parallelism=f"replicas x{world} (one time frame per GPU)",
                        l2="inputs larger than L2 (no flush needed)", inputs="device-resident, borrowed"),
            stage_ms=dict(zip(("S1_grid", "S2_neighbours", "S3_clean", "S4_start", "S5_tracklets", "total"),
                              (round(float(v), 4) for v in stage_ms))),
            roofline=dict(kernel="S2 neighbour finder: k_nf_plan + k_neighbours", bound="hbm", achieved=s2_gbs,
                          peak=peaks["hbm_gbs"], unit="GB/s", frac=s2_gbs / peaks["hbm_gbs"],
                          frac_of_nominal_8000=s2_gbs / 8000.0, traffic=ncu_traffic(args, N),
                          algorithmic_bytes=s2_bytes, peak_source=peaks["source"]),
            roofline_dominant=dict(kernel="S5 tracklets: k_tracklets<A,B,C1,C2> + k_track_gather", bound="alu", achieved=s5_tops, peak=alu_peak,
                                   unit="Tfp32op/s (no FMA)", frac=s5_tops / alu_peak, traffic=None, flops=flops,
                                   work=work),
            e2e=dict(value=e2e_value, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h, steps=e2e_steps,
                     ms_per_step=e2e_ms / e2e_steps, mode=e2e_mode,
                     serial_value=n_all * e2e_steps_serial / (e2e_serial_ms * 1e-3),
                     serial_ms_per_step=e2e_serial_ms / e2e_steps_serial, pipelined=pipe_res),
            selector=dict(stage_ms_S6=round(s6_ms, 4), stage_ms_S7_residuals=round(s7_ms, 4), stage_ms_S8_merge=round(s8_ms, 4), n_selected=counts_sel["n_selected"], n_sel_hits=counts_sel["n_sel_hits"],
                          note="S6 (SURVEY 8(f)-1) is outside the timed step; e2e_selected = serial step S1-S6 shipping the "
                               "selected tracks + owner instead of every tracklet",
                          e2e_selected=dict(value=n_all * e2e_steps_serial / (e2e_sel_serial_ms * 1e-3), unit=UNIT,
                                            ms_per_step=e2e_sel_serial_ms / e2e_steps_serial, d2h_bytes_per_step=d2h_sel,
                                            h2d_bytes_per_step=h2d, mode="serial, 1 context",
                                            streaming_value=(n_all * e2e_n / (e2e_sel_stream_ms * 1e-3) if e2e_sel_stream_ms else None),
                                            streaming_ms_per_step=(e2e_sel_stream_ms / e2e_n if e2e_sel_stream_ms else None))),
            gpu_launches=int(launches_per_step * args.steps),
            clocks=clocks, cpu_baseline=cpu, parity=parity, generate_s=round(gen_s, 1), footprint_4e8=footprint,
        )
        print(json.dumps(line), flush=True)
    trk.close()
    if world > 1:
        dist.destroy_process_group()


def launch_ranks(n):
    """`python bench.py --gpus N` without a launcher: start N ranks of this same command line, one per GPU, under
    torch.distributed.run on 127.0.0.1 (what the driver does itself for its scaling runs) and pass on the exit code.
    NCCL's communicator log stays on (NCCL_DEBUG=INFO, INIT subsystem, stderr) so the ranks can be counted."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.run(cmd, env=env).returncode


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tpcca", choices=["tpcca", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--mult-scale", type=float, default=1.0)
    ap.add_argument("--seed", type=int, default=None)
    ap.add_argument("--max-start-hits", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--ref-z-frac", type=float, default=0.25)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sectors", type=int, default=36, help="sectors the CPU baseline (the oracle) is timed on; default: all")
    ap.add_argument("--parity-sectors", type=int, default=8, help="sectors of the full-size parity check against the oracle")
    ap.add_argument("--footprint-scale", type=float, default=2.75,
                    help="mult_scale of the extra ~4e8-cluster footprint leg of the default workload (0: off)")
    ap.add_argument("--no-streaming", action="store_true", help="e2e with one context only")
    ap.add_argument("--pipeline-groups", type=int, default=3, help="sector groups of the tpcca_pipeline e2e leg (0/1: off)")
    ap.add_argument("--e2e-contexts", type=int, default=2, help="contexts (time frames in flight) of the streaming e2e mode")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "tpcca":
        args.warmup = 3        # timing rule: W >= 3
    return args


def main():
    args = parse_args()
    if "WORLD_SIZE" in os.environ:      # one line per rank on stderr: the launch can be counted from the log
        print(f"bench.py rank {os.environ.get('RANK', '0')}/{os.environ['WORLD_SIZE']} started (pid {os.getpid()}, "
              f"impl {args.impl})", file=sys.stderr, flush=True)
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(launch_ranks(args.gpus))
    else:
        run_tpcca(args)


if __name__ == "__main__":
    main()
