"""N > 1 on CPU: the path shards as independent replicas, so the only
cross-rank logic is bench.py's: per-rank seeds, MAX-over-ranks timing, rank 0 alone printing.
world_size-2 gloo processes on 127.0.0.1."""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        got = bench.max_over_ranks([1.0 + rank, 10.0 - rank, 5.0], dist, torch.device("cpu"))
        seeds = [bench.replica_seed(1, l, rank) for l in range(8)]
        gathered = [None] * world
        dist.all_gather_object(gathered, seeds)
        q.put((rank, got, gathered))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_replica_seeds_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, got, gathered in res:
        assert got == [2.0, 10.0, 5.0]                      # the slowest rank sets every time
        flat = [s for per_rank in gathered for s in per_rank]
        assert len(set(flat)) == len(flat)                  # no two (rank, layer) pairs share a batch


def test_reference_arm_under_two_ranks_prints_once():
    # `bench.py --impl reference` launched as 2 ranks: rank 0 prints the JSON line, rank 1 exits 0 silently
    outs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT="29400")
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["config"]["workload"].startswith("BASELINE.json configs[1]")
