"""N > 1 path of bench.py on CPU: two gloo processes (world_size 2).  The decoder does not shard a time frame
("replicas only"), so the only multi-rank logic is which time frame a rank decodes and how the per-rank
device times and cluster counts become the job's number: time = max over ranks, clusters = sum over ranks."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r "measured" (10 + 5 r) ms for (1000 + r) clusters
        ms, n = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000.0 + rank, torch.device("cpu"))
        # every rank draws its own time frame of the same recipe
        from tmd_inputs import build_geometry, timeframe as tf
        from tmd_inputs.physical import config2_like
        cfg = config2_like(300, 0, seed=3)
        cfg.seed += 1000 * bench.rank_seed_offset(rank)
        tr = tf.generate_truth(cfg, build_geometry(36), "cpu", batch=500)
        q.put((rank, ms, n, int(tr.n_attached), int(tr.att[:64].sum())))
    finally:
        dist.destroy_process_group()


def test_two_ranks_aggregate_max_time_and_sum_of_clusters():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, n, _, _ in got:
        assert ms == 15.0 and n == 2001.0          # max of (10, 15); 1000 + 1001
    assert got[0][3:] != got[1][3:]                # different time frames on the two ranks


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(3.5, 7.0, torch.device("cpu")) == (3.5, 7.0)


def test_bench_gpus_flag_starts_the_ranks_itself():
    # `python bench.py --gpus 2` outside torchrun must launch two ranks (torch.distributed.run on 127.0.0.1), not silently
    # run one: the rank plumbing is exercised on CPU with gloo (--rank-logic-only skips the CUDA work)
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--rank-logic-only"], capture_output=True,
                       text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                          # rank 0 alone prints
    assert lines[0]["n_gpus"] == 2 and lines[0]["ms_per_step"] == 15.0 and lines[0]["value"] == 2001.0 / 15e-3


def test_bench_refuses_a_world_size_that_contradicts_gpus():
    import subprocess
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--no-extras"], capture_output=True, text=True,
                       timeout=300, env=env)
    assert r.returncode != 0 and "WORLD_SIZE" in (r.stderr + r.stdout)
