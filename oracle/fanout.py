"""Process fan-out of oracle calls over independent units -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Every (tile) and every (sequence, KV head) unit of the KVarN path is independent, so the
slow float64 oracle can be spread over the host cores unit by unit.  Used by the parity tests (to afford the >= 1 %
samples SURVEY 8(d) asks for) and by bench.py's cpu_baseline (the all-core figure).  Holds no KVarN arithmetic: the
workers call oracle/kvarn_oracle.py as it stands.  Imports numpy only.
"""
from __future__ import annotations

import os

import numpy as np

_BLAS_ENV = ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS")


def n_cores() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


# ---- workers (top level: picklable under spawn) --------------------------------------------------------------
def _w_quantize(args):
    """One tile through the oracle quantizer, once free-running (trajectory, Alg. 1's own choice) and once at the
    iterate `at_k` the kernel kept (reading R10).  Returns plain arrays only."""
    from oracle import kvarn_oracle as O
    X, kind, bits, iters, rotate_on, aux_round, at_k = args
    X = np.asarray(X, dtype=np.float64)
    free = O.quantize_tile(X, kind, bits=bits, iters=iters, rotate_on=rotate_on, aux_round=aux_round)
    ref = free if (at_k is None or at_k == free.k_best) else \
        O.quantize_tile(X, kind, bits=bits, iters=iters, rotate_on=rotate_on, aux_round=aux_round, at_k=at_k)
    return {"I": np.array(free.varn.I), "k_free": free.k_best, "codes_free": free.codes,
            "codes": ref.codes, "s1": ref.s1, "s2": ref.s2, "z": ref.z,
            "s1_f": ref.s1_f, "s2_f": ref.s2_f, "z_f": ref.z_f}


def _w_decode(args):
    """Plain-definition attention of one (sequence, KV head) unit over stored tiles + raw tokens."""
    from oracle import kvarn_oracle as O
    q, kt, vt, kraw, vraw, sm_scale, rot_k, rot_v = args
    f = lambda t: tuple(np.asarray(a, dtype=np.float64) if i else a for i, a in enumerate(t))
    return O.decode_attention(np.asarray(q, dtype=np.float64), [f(t) for t in kt], [f(t) for t in vt],
                              np.asarray(kraw, dtype=np.float64), np.asarray(vraw, dtype=np.float64),
                              sm_scale=sm_scale, rotate_k=rot_k, rotate_v=rot_v)


def _w_cache_attention(args):
    """End to end for one unit: (attention over the oracle's OWN cache -- every chunk quantised by the oracle --,
    attention over the raw, un-quantised K and V)."""
    from oracle import kvarn_oracle as O
    q, K, V, n_sink, bits = args
    q, K, V = (np.asarray(a, dtype=np.float64) for a in (q, K, V))
    return O.cache_attention(q, K, V, n_sink=n_sink, bits=bits), O.attention(q, K, V)


def _w_decode_cycled(args):
    """Timing aid of bench.py's cpu_baseline: attention of one unit whose n_chunks chunks cycle through a few
    stored tiles (so the job is small to ship; the arithmetic is that of any unit of that length)."""
    from oracle import kvarn_oracle as O
    q, ks, vs, n_chunks = args
    kc = [ks[i % len(ks)] for i in range(n_chunks)]
    vc = [vs[i % len(vs)] for i in range(n_chunks)]
    return O.decode_attention(np.asarray(q, dtype=np.float64), kc, vc, np.zeros((0, q.shape[-1])), np.zeros((0, q.shape[-1])))


WORKERS = {"quantize": _w_quantize, "decode": _w_decode, "cache_attention": _w_cache_attention,
           "decode_cycled": _w_decode_cycled}


def _serve():
    """Worker process: (worker name, jobs) pickled on stdin -> results pickled on stdout."""
    import pickle
    import sys
    name, jobs = pickle.load(sys.stdin.buffer)
    fn = WORKERS[name]
    out = [fn(j) for j in jobs]
    pickle.dump(out, sys.stdout.buffer, protocol=pickle.HIGHEST_PROTOCOL)
    sys.stdout.buffer.flush()


def pmap(worker: str, jobs: list, procs: int | None = None) -> list:
    """[WORKERS[worker](j) for j in jobs], over `procs` worker processes (default: all cores), each with its BLAS
    pinned to one thread.  procs = 1 runs in this process (BLAS threads as they are).  The workers are fresh
    interpreters (`python -c ... _serve()`), fed through pipes: nothing of the parent -- its __main__, its CUDA
    context -- is inherited."""
    import pickle
    import subprocess
    import sys
    import threading
    fn = WORKERS[worker]
    procs = n_cores() if procs is None else max(1, int(procs))
    procs = min(procs, max(len(jobs), 1))
    if procs == 1:
        return [fn(j) for j in jobs]
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, PYTHONPATH=root + os.pathsep + os.environ.get("PYTHONPATH", ""))
    for k in _BLAS_ENV:
        env[k] = "1"                     # no BLAS oversubscription: one thread per worker
    shards = [list(range(i, len(jobs), procs)) for i in range(procs)]    # round-robin: even load
    ps = [subprocess.Popen([sys.executable, "-c", "from oracle.fanout import _serve; _serve()"], cwd=root, env=env,
                           stdin=subprocess.PIPE, stdout=subprocess.PIPE) for _ in shards]
    outs: list = [None] * procs

    def feed(i):
        data = pickle.dumps((worker, [jobs[j] for j in shards[i]]), protocol=pickle.HIGHEST_PROTOCOL)
        outs[i], _ = ps[i].communicate(data)

    th = [threading.Thread(target=feed, args=(i,)) for i in range(procs)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    res: list = [None] * len(jobs)
    for i, pr in enumerate(ps):
        if pr.returncode != 0:
            raise RuntimeError(f"oracle fan-out worker {i} exited with {pr.returncode}")
        for j, r in zip(shards[i], pickle.loads(outs[i])):
            res[j] = r
    return res
