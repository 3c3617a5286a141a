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
