"""N > 1 host logic of bench.py on CPU: world_size 2, `gloo` backend.

The hot path shards with no data-path collective (one time frame per GPU), so what N > 1 adds is host
logic only: a distinct seeded time frame per rank, the max-over-ranks of the device time, the sum of the
processed clusters, and rank-0-only printing.  No CUDA here; the kernels are covered by the -m gpu tests.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    import tpcsynth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cpu")
    seed = bench.rank_seed(0, None, rank)
    tf = tpcsynth.generate(0, seed=seed)
    ms_local = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    value, ms, n_all = bench.whole_job_value(tf.n_clusters, 4, ms_local, world, dev)
    gathered = [None] * world
    dist.all_gather_object(gathered, (seed, tf.n_clusters, float(tf.y[0][:8].sum())))
    if rank == 0:
        out.put(dict(value=value, ms=ms, n_all=n_all, gathered=gathered))
    dist.destroy_process_group()


def test_replicas_world2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (s0, n0, c0), (s1, n1, c1) = res["gathered"]
    import tpcsynth
    assert s0 == tpcsynth.generator.BASE_SEED and s1 == s0 + 1000       # rank 0 keeps BASELINE.json's seed
    assert c0 != c1                                                       # different time frames per rank
    assert res["ms"] == 15.0                                              # max over ranks
    assert res["n_all"] == n0 + n1                                        # whole-job units
    assert np.isclose(res["value"], (n0 + n1) * 4 / 15.0e-3)


def test_reference_arm_prints_on_rank0_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 prints the line, rank 1 exits 0 silently."""
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--config", "0", "--ref-z-frac", "1.0"]
    r1 = subprocess.run(cmd, env=dict(env, RANK="1", LOCAL_RANK="1"), capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(env, RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["n_gpus"] == 2


# ------------------------------------------------------------------------------------------------
# run_tpcca's own N > 1 branch (process group, barriers, reductions, rank-0 line) with the device side
# replaced by a CPU stand-in at the Tracker / torch.cuda boundary
# ------------------------------------------------------------------------------------------------
class _FakeView:
    def __init__(self, n):
        self.n_clusters, self.n_start, self.n_tracks, self.n_hits = n, n // 30, n // 40, n // 2
        self.n_selected, self.n_sel_hits = n // 160, n // 8


class _FakeTracker:
    """Stands in for paper_2208_07412_b200.Tracker: no compute, a simulated device clock."""
    def __init__(self, env, params):
        self.env, self.n = env, 0

    def reset(self):
        self.n = 0
        self.sec = []

    def load_clusters(self, s, y, z, row, borrow=False):
        self.sec.append(int(y.shape[0])); self.n += int(y.shape[0])

    def run(self, mask=31):
        self.env.clock_ms += self.env.step_ms

    def sync(self):
        pass

    def launch_count(self):
        return 30

    def counts(self):
        return dict(n_clusters=self.n, n_start=self.n // 30, n_tracks=self.n // 40, n_hits=self.n // 2, n_bins=1000,
                    n_selected=self.n // 160, n_sel_hits=self.n // 8)

    def timings(self, i=0):
        t = self.env.step_ms
        return [0.1 * t, 0.1 * t, 0.05 * t, 0.05 * t, 0.7 * t, t, 0.02 * t, 0.01 * t, 0.01 * t]

    def work_counters(self):
        return dict(propagations=10, updates=10, gates=1, searches=5, candidates=9)

    def get_tracks_view(self, s, mem, what):
        return _FakeView(self.sec[s])

    def get_tracks_all_views(self, mem, what):
        return [_FakeView(n) for n in self.sec]

    def close(self):
        pass


class _FakeEvent:
    def __init__(self, env):
        self.env, self.t = env, 0.0

    def record(self):
        self.t = self.env.clock_ms

    def elapsed_time(self, other):
        return other.t - self.t


class FakeEnv:
    backend = "gloo"
    oom_error = MemoryError

    def __init__(self, rank, world, local):
        from paper_2208_07412_b200 import binding as B     # constants only; no library call
        self.B = B
        self.device = torch.device("cpu")
        self.clock_ms = 0.0
        self.step_ms = 10.0 + 5.0 * rank                   # rank 1 is the slow one
        self.rank = rank

    def init_process_group(self):
        dist.init_process_group(self.backend)

    def tracker(self, params, max_clusters, max_start_hits, stream=None):
        return _FakeTracker(self, params)

    def pipeline(self, *a):
        raise AssertionError("the pipeline leg runs at N = 1 only")

    def pin(self, a):
        return torch.from_numpy(a)

    def pin_u16(self, a):
        return torch.from_numpy(a.view(np.int16))

    def to_device(self, t):
        return t

    def event(self):
        return _FakeEvent(self)

    def synchronize(self):
        pass

    def set_thread_device(self):
        pass

    def stream(self):
        return object()

    def wait_stream(self, sd):
        pass

    def empty_cache(self):
        pass

    def sm_count(self):
        return 148

    def clock_sampler(self):
        class _S:
            def start(self): pass
            def stop(self, a, b): return dict(sm_mhz=None, sm_max_mhz=None, reasons=["stub"])
        return _S()


def _bench_worker(rank, world, port, out):
    import contextlib
    import io
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import bench
    from test_multirank import FakeEnv
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    sys.argv = ["bench.py", "--gpus", str(world), "--steps", "4", "--warmup", "3", "--config", "0"]
    buf = io.StringIO()
    with contextlib.redirect_stdout(buf):
        args = bench.parse_args()
        bench.run_tpcca(args, FakeEnv)
    out.put((rank, buf.getvalue()))


def test_run_tpcca_world2_with_stub_device():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_bench_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(out.get(timeout=180) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[1].strip() == ""                                      # only rank 0 prints
    line = json.loads(got[0].strip().splitlines()[-1])
    import tpcsynth
    n0 = tpcsynth.generate(0).n_clusters
    n1 = tpcsynth.generate(0, seed=tpcsynth.generator.BASE_SEED + 1000).n_clusters
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and line["steps"] == 4
    assert line["config"]["n_clusters_per_gpu"] == n0 and "replicas x2" in line["config"]["parallelism"]
    assert abs(line["ms_per_step"] - 15.0) < 1e-9                    # max over ranks of the device time
    assert np.isclose(line["value"], (n0 + n1) * 4 / (4 * 15.0e-3))  # whole-job clusters / slowest rank's time
    assert line["cpu_baseline"] is None and line["e2e"]["value"] > 0


def test_bench_gpus_n_starts_n_ranks():
    """`python bench.py --gpus 2` with no launcher in the environment starts ranks 0 and 1 itself; without a GPU
    each fails loudly (there is no CPU path) and the launcher passes the failure on."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env["CUDA_VISIBLE_DEVICES"] = ""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--config", "0"],
                       env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode != 0
    assert "bench.py rank 0/2 started" in r.stderr and "bench.py rank 1/2 started" in r.stderr
    assert "needs a CUDA device: tpcca has no CPU path" in r.stderr     # (the launcher stops the other rank at the first failure)
