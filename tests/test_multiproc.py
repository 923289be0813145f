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


def _cp_worker(rank, world, port, q):
    """Context-parallel merge on CPU tensors: every rank computes the oracle's partial {m, l, o} of its chunk share
    (bench.cp_shard), all-gathers them with gloo and merges -- the result must equal attention over the whole sequence."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import numpy as np
    import bench
    from oracle import kvarn_oracle as O
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(7)
        n_chunks, g = 5, 4
        K = rng.standard_normal((n_chunks * 128 + 9, 128)); V = rng.standard_normal((n_chunks * 128 + 9, 128))
        qh = rng.standard_normal((g, 128))
        lo, hi = bench.cp_shard(n_chunks, rank, world)
        t0, t1 = lo * 128, hi * 128 + (9 if rank == world - 1 else 0)
        logits = (qh @ K[t0:t1].T) / np.sqrt(128) * np.log2(np.e)          # log2 units, like the kernel's partials
        m = logits.max(axis=1) if t1 > t0 else np.full(g, -np.inf)
        p = np.exp2(logits - m[:, None])
        part = torch.tensor(np.concatenate([m[:, None], p.sum(1)[:, None], np.zeros((g, 2)), p @ V[t0:t1]], axis=1))
        parts = [torch.empty_like(part) for _ in range(world)]
        dist.all_gather(parts, part)
        P = torch.stack(parts).numpy()
        mstar = P[:, :, 0].max(axis=0)
        w = np.exp2(P[:, :, 0] - mstar[None])
        out = (w[:, :, None] * P[:, :, 4:]).sum(0) / (w * P[:, :, 1]).sum(0)[:, None]
        ref = O.attention(qh, K, V)
        q.put((rank, float(np.abs(out - ref).max()), (lo, hi)))
    finally:
        dist.destroy_process_group()


def test_context_parallel_shards_and_lse_merge_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29700 + os.getpid() % 2000
    procs = [ctx.Process(target=_cp_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert [r[2] for r in res] == [(0, 3), (3, 5)]           # contiguous shares, sizes differ by at most one
    assert all(r[1] < 1e-12 for r in res)


def test_cp_shard_covers_every_chunk_once():
    sys.path.insert(0, ROOT)
    import bench
    for n in (0, 1, 7, 512):
        for world in (1, 2, 3, 8):
            spans = [bench.cp_shard(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            assert max(h - l for l, h in spans) - min(h - l for l, h in spans) <= 1
