#!/usr/bin/env python
"""bench.py -- KVarN hot path on B200: BASELINE.json configs[1] (Llama-3.1-8B-
shaped decode layer: B=8, 32 q / 8 KV heads, head_dim 128, ctx 8192 = 64 chunks,
2-bit), one JSON line.

A "step" is one pass of the whole hot path over one batch of synthetic input:
  write path  kvarn_quantize_chunk over the batch's 2 x 4096 K/V tiles (one launch)
  read path   kvarn_decode_attention over a 64-chunk packed cache (one launch: the split
              partials merge inside the kernel through DSMEM of a thread-block cluster)
The bench cycles through L = 8 distinct "layers" (input + cache copies, 2.4 GB
of inputs, 302 MB of records: far larger than the 126 MB L2); the read path of
step i reads the cache written L/2 steps earlier, so neither kernel ever finds
its input in L2.  Each kernel is timed with CUDA events on the launching
stream inside the timed region.

  metric/value  2-bit decode-attention GB/s  (algorithmic bytes / decode time)
  also          quantize tokens/s, us/step, HBM / ALU roofline fractions,
                the oracle timed on the host cores (cpu_baseline), the same step through
                the host-buffer C-ABI calls (e2e), and -- at N = 1 -- the long-context
                (configs[4]-shaped) decode and the configs[3] quantizer sweep ("extras").

`--impl reference` times the CPU oracle (oracle/) on a bounded sample instead.
Under torchrun (N > 1) every rank runs an independent replica of the workload
(the path has no cross-sequence exchange: DESIGN.md "Multi-GPU").
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
import torch

D, G = 128, 128
FP32_PEAK_TFLOPS_NOMINAL = 148 * 128 * 2 * 1.965e9 / 1e12  # SMs x lanes x FMA x max clock
# Algorithmic fp32 flops of the write path per tile:
#   Hadamard 7 stages x 16384 add/sub                       = 114 688
#   Alg. 1, K=8: 18 variance passes x 16384 x (mul+add+fma) = 1 179 648  (4 flop / element / pass)
#   balance (2 mul) + RTN (min, max, fma, round, 2 clamp)    =   131 072
QUANT_FLOPS_PER_TILE = 7 * 16384 + 18 * 16384 * 4 + 8 * 16384


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def tensor_peak():
    """Dense bf16 / fp16 tensor throughput in TFLOP/s: the measured burst figure, else the guide's nominal 2250."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        if d.get("bf16_tflops"):
            return float(d["bf16_tflops"]), "measured burst (MEASURED_PEAKS.json bf16_tflops; fp16 = bf16 rate)"
    return 2250.0, "fallback (nominal dense bf16, B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(index)], stdout=subprocess.PIPE, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except Exception:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(smax)) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _blas_one_thread():
    """Context manager pinning numpy's BLAS to one thread (threadpoolctl is in the image)."""
    from threadpoolctl import threadpool_limits
    return threadpool_limits(limits=1)


def oracle_inputs(n_tiles: int, g: int, seed: int = 1):
    """n_tiles K and V tiles of the configs[1] recipe + g query heads, as float32 / float64 numpy arrays."""
    from paper_2606_03458_b200 import workloads as W
    K, V = W.kv_tokens(1, 1, n_tiles * G, seed=seed, device="cpu")
    q = W.queries(1, g, seed=seed, device="cpu")[0].double().numpy()
    return K[0, 0].float().numpy().reshape(n_tiles, G, D), V[0, 0].float().numpy().reshape(n_tiles, G, D), q


def oracle_sample(n_tiles: int, n_units: int, n_chunks: int, g: int, procs: int = 1, seed: int = 1):
    """Time the oracle, as it stands, on a bounded sample of configs[1]: quantize_tile on n_tiles K + n_tiles V
    tiles, then decode_attention of n_units (sequence, KV head) units over n_chunks chunks each (the units' chunk
    lists cycle through the quantised tiles).  procs = 1: in this process with BLAS pinned to one thread;
    procs > 1: oracle/fanout.py spreads the independent tiles / units over that many single-threaded processes.
    Returns (seconds for the tiles, seconds for the units)."""
    from oracle import fanout
    Kt, Vt, q = oracle_inputs(n_tiles, g, seed)
    jobs = [(x, "k", 2, 8, True, "after", None) for x in Kt] + [(x, "v", 2, 8, True, "after", None) for x in Vt]
    with _blas_one_thread():
        t0 = time.perf_counter()
        res = fanout.pmap("quantize", jobs, procs)
        t_q = time.perf_counter() - t0
        ks = [(r["codes"], r["s1"], r["s2"], r["z"]) for r in res[:n_tiles]]
        vs = [(r["codes"], r["s1"], r["s2"], r["z"]) for r in res[n_tiles:]]
        ks, vs = ks[:8], vs[:8]        # the units cycle through (at most) 8 distinct tiles: small jobs to ship
        t0 = time.perf_counter()
        fanout.pmap("decode_cycled", [(q, ks, vs, n_chunks)] * n_units, procs)
        t_d = time.perf_counter() - t0
    return t_q, t_d


def cpu_baseline_both(shape, rb, budget_s: float = 6.0):
    """cpu_baseline of the JSON line: the oracle on one thread and fanned over all host cores (BASELINE.md's plan),
    each on a sample sized for ~budget_s seconds per half (probed first on this host)."""
    from oracle import fanout
    cores = fanout.n_cores()
    unit_bytes = shape.n_chunks * 2 * rb + shape.g * (D * 2 + D * 4)
    pq, pd = oracle_sample(4, 1, shape.n_chunks, shape.g, 1)
    out = {}
    for name, procs in (("one_thread", 1), ("all_cores", cores)):
        n_t = int(min(max(procs * budget_s / max(pq / 8, 1e-4), 8), 8192))
        n_u = int(min(max(procs * budget_s / max(pd, 1e-3), 2), 2048))
        tq, td = oracle_sample(n_t, n_u, shape.n_chunks, shape.g, procs)
        out[name] = {"cores": procs, "decode_GBps": sig(n_u * unit_bytes / td / 1e9), "quantize_tokens_per_s": sig(n_t * G / tq / shape.Hkv),
                     "tiles": 2 * n_t, "tiles_s": sig(tq), "units": n_u, "units_s": sig(td)}
    best = out["all_cores"]
    return {"value": best["decode_GBps"], "unit": "GB/s", "cores": cores, "kind": "oracle",
            "sample": f"numpy f64 oracle, {cores} single-threaded processes: quantize_tile on {best['tiles']} tiles, decode_attention on "
                      f"{best['units']} (seq, KV head) units x {shape.n_chunks} chunks",
            "quantize_tokens_per_s": best["quantize_tokens_per_s"], "one_thread": out["one_thread"], "all_cores": out["all_cores"]}


def run_reference(args, shape):
    """--impl reference: the oracle on the host cores (all of them, one single-threaded process each), same metric
    and config as the kvarn arm; every step is a bounded sample of the workload."""
    from oracle import fanout
    cores = fanout.n_cores()
    pq, pd = oracle_sample(4, 1, shape.n_chunks, shape.g, 1)
    budget = min(3.0, 60.0 / (2 * max(args.steps + min(args.warmup, 1), 1)))   # seconds per half-step: whole run ~ 1 min
    n_tiles = int(min(max(cores * budget / max(pq / 8, 1e-4), 8), 4096))
    n_units = int(min(max(cores * budget / max(pd, 1e-3), 2), 1024))
    rec_bytes = 4608
    unit_bytes = shape.n_chunks * 2 * rec_bytes + shape.g * (D * 2 + D * 4)
    for _ in range(min(args.warmup, 1)):
        oracle_sample(8, 2, 4, shape.g, cores)
    tq = td = 0.0
    t_all = time.perf_counter()
    for _ in range(args.steps):
        a, b = oracle_sample(n_tiles, n_units, shape.n_chunks, shape.g, cores)
        tq += a; td += b
    wall = time.perf_counter() - t_all
    gbs = n_units * unit_bytes * args.steps / td / 1e9
    tok_s = n_tiles * G * args.steps / tq / shape.Hkv   # a token = one position across the 8 KV heads, K and V
    sample = (f"per step: quantize_tile on {2 * n_tiles} tiles, decode_attention on {n_units} (seq, KV head) units x "
              f"{shape.n_chunks} chunks; numpy f64 oracle over {cores} single-threaded processes")
    line = {
        "impl": "reference", "metric": "kvarn_2bit_decode_attn_GBps", "value": sig(gbs), "unit": "GB/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": sig(wall / args.steps * 1e3), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(shape, args.layers),
        "quantize_tokens_per_s": sig(tok_s),
        "cpu_baseline": {"value": sig(gbs), "unit": "GB/s", "cores": cores, "kind": "oracle",
                         "sample": sample, "quantize_tokens_per_s": sig(tok_s)},
        "e2e": {"value": sig(gbs), "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def sig(x, n: int = 4):
    """round to n significant digits (keeps the JSON line short enough for the driver's log tail)"""
    if x is None or isinstance(x, (str, bool, int)):
        return x
    x = float(x)
    if x == 0 or not np.isfinite(x):
        return x
    return float(f"{x:.{n}g}")


def compact(o):
    if isinstance(o, dict):
        return {k: compact(v) for k, v in o.items()}
    if isinstance(o, (list, tuple)):
        return [compact(v) for v in o]
    return sig(o)


def max_over_ranks(values, dist, device):
    """MAX over ranks of a list of floats (device times): the slowest replica sets the job's time."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def replica_seed(base: int, layer: int, rank: int) -> int:
    """Seed of layer `layer` of replica `rank`: every rank draws its own synthetic batch."""
    return base + 100 * layer + 1000 * rank


def workload_config(shape, layers, eager=False):
    return {"workload": "BASELINE.json configs[1]: Llama-3.1-8B-shaped decode layer",
            "B": shape.B, "Hq": shape.Hq, "Hkv": shape.Hkv, "head_dim": D, "ctx": shape.ctx,
            "chunks": shape.n_chunks, "resid": shape.resid, "bits": shape.bits,
            "step": "kvarn_quantize_chunk(2x%d tiles) of one layer + kvarn_decode_attention of all %d layers (one launch per layer%s)"
                    % (shape.B * shape.Hkv * shape.n_chunks, layers, "" if eager else ", replayed as one CUDA graph"),
            "l2": "inputs larger than L2: %d layer caches read in rotation (%d MB of records per step)"
                  % (layers, layers * 2 * shape.B * shape.Hkv * shape.n_chunks * 4608 // 1000000),
            "parallelism": "replicas"}


def _time_launches(fn, n, stream):
    """median / min device time (ms) of n launches of fn(i), CUDA events on the launching stream"""
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
    for i in range(n):
        evs[i][0].record(stream); fn(i); evs[i][1].record(stream)
    torch.cuda.synchronize()
    ts = sorted(a.elapsed_time(b) for a, b in evs)
    return ts[len(ts) // 2], ts[0]


def _fill_cache(kv, W, p, sh, dev, n_sink=0, max_chunks=None):
    cache = kv.Cache(p, sh.B, sh.Hkv, sh.n_chunks if max_chunks is None else max_chunks, device=dev, n_sink=n_sink)
    for b0 in range(0, sh.B, 4):   # fill 4 sequences at a time (1.1 GB of bf16 K/V each at 64k tokens)
        K, V = W.kv_tokens(4, sh.Hkv, sh.ctx, seed=sh.seed + b0, device=dev)
        kv.prefill(p, cache.slice(b0, b0 + 4), K, V)
        del K, V
    return cache


def run_extras(kv, W, dev, hbm_peak, only=frozenset()):
    """The other configs, one B200 (N = 1 only).  Groups (select with --extras-only --only a,b):
      decode  = cfg4 + long.  cfg4: configs[4] (B=64, 64 q / 8 KV heads, ctx 65536 + 64 residual), 2-bit and 4-bit;
              long: a 64k-context g = 4 cache (B=16, 32/8 heads), 2-bit and 4-bit, + block attention (n_q = 2, 8) and
              kvarn_append_block on it
      sink    the same g = 4 cache in the paper's three-region layout with S = 128 raw sink tokens
      cfg2    configs[2]: the last 256 steps of the growth to 32768 tokens, one append + one decode per step
      quant   configs[3]: 8 heads x 2^20 tokens in one launch, 2-bit and 4-bit; the paper's 576-tile latency case
      rot     RoPE + Hadamard of 2^18 tokens x 8 heads (App. A)
    Launches that read more than L2 holds are simply repeated; short launches are timed inside CUDA graphs."""
    stream = torch.cuda.current_stream()
    want = lambda g: not only or g in only
    ex = {}
    if want("decode") or want("cfg4") or want("long"):
        long_g4 = W.DecodeShape("long_context_g4", B=16, Hq=32, Hkv=8, ctx=65536, seed=5)   # Llama-3.1-8B heads, 64k context
        shapes = [("decode_cfg4", W.CONFIG4)] * (want("decode") or want("cfg4")) + [("decode_long_g4", long_g4)] * (want("decode") or want("long"))
        for name, sh in shapes:
            for bits in (2, 4):
                p = kv.default_params(bits)
                cache = _fill_cache(kv, W, p, sh, dev)
                q = W.queries(sh.B, sh.Hq, seed=sh.seed, device=dev)
                ws = torch.empty((max(kv.decode_workspace_bytes(p, sh.B, sh.Hq, sh.Hkv, sh.n_chunks), 16),), dtype=torch.uint8, device=dev)
                out = torch.empty((sh.B, sh.Hq, D), dtype=torch.float32, device=dev)
                for _ in range(3):
                    kv.decode_attention(p, cache, q, out=out, ws=ws)
                torch.cuda.synchronize()
                med, mn = _time_launches(lambda i: kv.decode_attention(p, cache, q, out=out, ws=ws), 10, stream)
                byts = cache.nbytes_read_by_decode(sh.ctx) + sh.B * sh.Hq * (D * 2 + D * 4)
                ex[f"{name}_{bits}bit"] = {"us": med * 1e3, "GBps": byts / med / 1e6, "hbm_frac": byts / med / 1e6 / hbm_peak,
                                           "MB": byts / 1e6, "shape": f"B{sh.B} {sh.Hq}/{sh.Hkv} ctx{sh.ctx}"}
                if bits == 2:
                    # the same launch with 16-bit q~ (kvarn_params::decode_digits = 2: half the QK^T tensor-core work; its
                    # error is statistically ~3e-4 but has no deterministic bound below the 2e-3 tolerance: not the default)
                    p2 = kv.default_params(bits)
                    p2.decode_digits = 2
                    for _ in range(3):
                        kv.decode_attention(p2, cache, q, out=out, ws=ws)
                    torch.cuda.synchronize()
                    med2, _ = _time_launches(lambda i: kv.decode_attention(p2, cache, q, out=out, ws=ws), 10, stream)
                    ex[f"{name}_{bits}bit_digits2"] = {"us": med2 * 1e3, "GBps": byts / med2 / 1e6, "hbm_frac": byts / med2 / 1e6 / hbm_peak}
                if name == "decode_long_g4" and bits == 2:
                    # multi-token read path (Fig. 4): a block of n_q new tokens against the same cache
                    for n_q in (2, 8):
                        qb = torch.stack([W.queries(sh.B, sh.Hq, seed=sh.seed + 100 + i, device=dev) for i in range(n_q)], dim=1).contiguous()
                        kb, vb = W.kv_tokens(sh.B, sh.Hkv, n_q, seed=sh.seed + 200, device=dev, sink_first=False)
                        ob = torch.empty((sh.B, n_q, sh.Hq, D), dtype=torch.float32, device=dev)
                        for _ in range(3):
                            kv.block_attention(p, cache, qb, kb, vb, out=ob)
                        torch.cuda.synchronize()
                        medb, _ = _time_launches(lambda i: kv.block_attention(p, cache, qb, kb, vb, out=ob), 10, stream)
                        bb = cache.nbytes_read_by_decode(sh.ctx) + sh.B * n_q * (sh.Hq * (D * 2 + D * 4) + 2 * sh.Hkv * D * 2)
                        ex[f"block_long_g4_2bit_nq{n_q}"] = {"us": medb * 1e3, "us_per_query_token": medb * 1e3 / n_q,
                                                             "hbm_frac": bb / medb / 1e6 / hbm_peak, "x_decode": medb / med}
                        if n_q == 8:
                            # write half of the pseudo-decode step: the block joins the cache (13 x 8 tokens fit the residual window)
                            meda, _ = _time_launches(lambda i: kv.append_block(p, cache, kb, vb), 13, stream)
                            ex["append_block_nq8"] = {"us": meda * 1e3, "note": "8 tokens x 16 sequences, one launch"}
                        del qb, kb, vb, ob
                if name == "decode_long_g4":
                    # the dense tcgen05 form of the same call (kvarn_block_attention_dense) on blocks of 8, 32 and 128 tokens
                    for n_q in ((8, 32, 128) if bits == 2 else (32,)):
                        qb = torch.stack([W.queries(sh.B, sh.Hq, seed=sh.seed + 100 + i, device=dev) for i in range(n_q)], dim=1).contiguous()
                        kb, vb = W.kv_tokens(sh.B, sh.Hkv, n_q, seed=sh.seed + 200, device=dev, sink_first=False)
                        ob = torch.empty((sh.B, n_q, sh.Hq, D), dtype=torch.float32, device=dev)
                        wsd = torch.empty((int(kv.lib.kvarn_block_dense_workspace_bytes(p, sh.B, sh.Hq, sh.Hkv, n_q, sh.n_chunks)),),
                                          dtype=torch.uint8, device=dev)
                        for _ in range(2):
                            kv.block_attention(p, cache, qb, kb, vb, out=ob, dense=True, ws=wsd)
                        torch.cuda.synchronize()
                        medd, _ = _time_launches(lambda i: kv.block_attention(p, cache, qb, kb, vb, out=ob, dense=True, ws=wsd), 5, stream)
                        flop = 4.0 * sh.B * sh.Hq * n_q * sh.ctx * D                      # QK^T + PV, 2 flop per MAC
                        tf = flop / (medd * 1e-3) / 1e12
                        ex[f"block_dense_long_g4_{bits}bit_nq{n_q}"] = {"us": medd * 1e3, "us_per_query_token": medd * 1e3 / n_q, "x_decode": medd / med,
                                                                   "TFLOPs": tf, "tensor_frac": tf / tensor_peak()[0],
                                                                   "note": "whole call: block_dense_kernel (packed chunks + raw windows) + merge; "
                                                                           "flop = 4 B Hq n_q ctx 128 (the hi / lo q terms are not counted twice)"}
                        del qb, kb, vb, ob, wsd
                del cache, q, ws, out
                torch.cuda.empty_cache()
    if want("sink"):
        # the paper's three-region layout: S = 128 raw sink tokens in front of the quantised body
        sh = W.DecodeShape("long_context_g4_sink128", B=16, Hq=32, Hkv=8, ctx=128 + 65536 + 64, seed=6)
        p = kv.default_params(2)
        cache = _fill_cache(kv, W, p, sh, dev, n_sink=128, max_chunks=512)
        q = W.queries(sh.B, sh.Hq, seed=sh.seed, device=dev)
        ws = torch.empty((max(kv.decode_workspace_bytes(p, sh.B, sh.Hq, sh.Hkv, 512), 16),), dtype=torch.uint8, device=dev)
        out = torch.empty((sh.B, sh.Hq, D), dtype=torch.float32, device=dev)
        for _ in range(3):
            kv.decode_attention(p, cache, q, out=out, ws=ws)
        torch.cuda.synchronize()
        med, mn = _time_launches(lambda i: kv.decode_attention(p, cache, q, out=out, ws=ws), 10, stream)
        byts = cache.nbytes_read_by_decode(sh.ctx) + sh.B * sh.Hq * (D * 2 + D * 4)
        ex["decode_long_g4_2bit_sink128"] = {"us": med * 1e3, "GBps": byts / med / 1e6, "hbm_frac": byts / med / 1e6 / hbm_peak}
        del cache, q, ws, out
        torch.cuda.empty_cache()
    if want("cfg2"):
        # configs[2] (Qwen3-4B-shaped incremental decode, B=16): the last 256 steps of the growth to 32768 tokens,
        # one kvarn_append + one kvarn_decode_attention per step (two chunk boundaries inside); 302 MB of records
        s2 = W.CONFIG2
        p = kv.default_params(2)
        n0 = s2.ctx - 256
        cache = kv.Cache(p, s2.B, s2.Hkv, s2.n_chunks, device=dev)
        K, V = W.kv_tokens(s2.B, s2.Hkv, s2.ctx, seed=s2.seed, device=dev)
        kv.prefill(p, cache, K[:, :, :n0].contiguous(), V[:, :, :n0].contiguous())
        q = W.queries(s2.B, s2.Hq, seed=s2.seed, device=dev)
        ws = torch.empty((max(kv.decode_workspace_bytes(p, s2.B, s2.Hq, s2.Hkv, s2.n_chunks), 16),), dtype=torch.uint8, device=dev)
        out = torch.empty((s2.B, s2.Hq, D), dtype=torch.float32, device=dev)
        Kt = K[:, :, n0:].permute(2, 0, 1, 3).contiguous()   # [256][B][Hkv][128]
        Vt = V[:, :, n0:].permute(2, 0, 1, 3).contiguous()
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(256)]
        for i in range(256):
            evs[i][0].record(stream); kv.append(p, cache, Kt[i], Vt[i])
            evs[i][1].record(stream); kv.decode_attention(p, cache, q, out=out, ws=ws)
            evs[i][2].record(stream)
        torch.cuda.synchronize()
        ap = [e[0].elapsed_time(e[1]) * 1e3 for e in evs]
        dc = [e[1].elapsed_time(e[2]) * 1e3 for e in evs]
        bnd = [i for i in range(256) if (n0 + i + 1) % G == 0]
        plain = sorted(ap[i] for i in range(8, 256) if i not in bnd)
        byts = cache.nbytes_read_by_decode(s2.ctx - 128) + s2.B * s2.Hq * (D * 2 + D * 4)
        dmed = sorted(dc[8:])[len(dc[8:]) // 2]
        final_len = int(cache.seq_lens[0].item())
        # the same 96 plain steps (no boundary inside: residual 1..96) replayed as ONE CUDA graph: append + decode back to back
        kv.prefill(p, cache, K[:, :, :n0].contiguous(), V[:, :, :n0].contiguous())
        fns = []
        for i in range(96):
            fns.append(lambda i=i: kv.append(p, cache, Kt[i], Vt[i]))
            fns.append(lambda: kv.decode_attention(p, cache, q, out=out, ws=ws))
        step_graph_us = 2 * _time_graph(fns, stream, replays=1, warm=False) * 1e3
        ex["cfg2_incremental"] = {"append_plain_us": plain[len(plain) // 2], "append_boundary_us": [ap[i] for i in bnd],
                                  "decode_us": dmed, "step_us": dmed + plain[len(plain) // 2], "step_graph_us": step_graph_us,
                                  "decode_GBps": byts / dmed / 1e3, "decode_hbm_frac": byts / dmed / 1e3 / hbm_peak,
                                  "step_graph_hbm_frac": byts / step_graph_us / 1e3 / hbm_peak,
                                  "ctx": [n0, s2.ctx], "final_seq_len": final_len,
                                  "note": "event pairs around single launches; step_graph = append + decode of 96 plain steps in one CUDA graph"}
        del cache, K, V, Kt, Vt, q, ws, out
        torch.cuda.empty_cache()
    if want("quant"):
        n_tok = 1 << 20
        K, V = W.quantizer_sweep_tiles(8, n_tok, seed=3, device=dev)
        n_tiles = 8 * n_tok // G
        Kt, Vt = K.view(n_tiles, G, D), V.view(n_tiles, G, D)
        for bits in (2, 4):
            p = kv.default_params(bits)
            rb = kv.record_bytes(p)
            kr = torch.empty((n_tiles, rb), dtype=torch.uint8, device=dev); vr = torch.empty_like(kr)
            for _ in range(2):
                kv.quantize_chunk(p, Kt, Vt, kr, vr)
            torch.cuda.synchronize()
            med, mn = _time_launches(lambda i: kv.quantize_chunk(p, Kt, Vt, kr, vr), 5, stream)
            byts = 2 * n_tiles * (G * D * 2 + rb)
            ex[f"quantize_cfg3_{bits}bit"] = {"ms": med, "tokens_per_s": n_tok / (med * 1e-3), "tiles_per_s": 2 * n_tiles / (med * 1e-3),
                                              "hbm_frac": byts / med / 1e6 / hbm_peak,
                                              "alu_frac": 2 * n_tiles * QUANT_FLOPS_PER_TILE / (med * 1e-3) / 1e12 / FP32_PEAK_TFLOPS_NOMINAL}
            del kr, vr
        # the paper's own write-path measurement (Sec. 4.2): "8 iterations of variance-normalization in every
        # attention layer in Qwen3-4B" for one 128-token chunk = 36 layers x 8 KV heads x {K, V} = 576 tiles, one launch.
        # Paper: 1.9 ms on "a GPU with 500 TFLOP at fp16 and 1.8 TB/s" (normalisation only; ours is the whole record). Context only.
        n_lat = 36 * 8
        p = kv.default_params(2)
        rb = kv.record_bytes(p)
        kr = torch.empty((n_lat, rb), dtype=torch.uint8, device=dev); vr = torch.empty_like(kr)
        srcs = [(Kt[i * n_lat:(i + 1) * n_lat], Vt[i * n_lat:(i + 1) * n_lat]) for i in range(64)]   # 64 distinct inputs (> L2 in total)
        for i in range(3):
            kv.quantize_chunk(p, srcs[i][0], srcs[i][1], kr, vr)
        torch.cuda.synchronize()
        med, mn = _time_launches(lambda i: kv.quantize_chunk(p, srcs[i % 64][0], srcs[i % 64][1], kr, vr), 64, stream)
        ex["quantize_latency_qwen3_4b_chunk"] = {"us": med * 1e3, "tiles": 2 * n_lat, "paper_ms_other_hw": 1.9}
        del kr, vr, Kt, Vt, K, V, srcs
        torch.cuda.empty_cache()
    if want("rot"):
        # App. A online transform fused with RoPE: K of 2^18 tokens x 8 heads, bf16; streaming kernel
        n_rt, h_rt = 1 << 18, 8
        xk = torch.randn((n_rt, h_rt, D), device=dev, dtype=torch.bfloat16)
        ang = torch.arange(n_rt, device=dev, dtype=torch.float32)[:, None] * (10000.0 ** (-torch.arange(0, D, 2, device=dev, dtype=torch.float32) / D))[None, :]
        ct, st = torch.cos(ang).contiguous(), torch.sin(ang).contiguous()
        yk = torch.empty_like(xk)
        for _ in range(2):
            kv.rope_hadamard(xk, ct, st, out=yk)
        torch.cuda.synchronize()
        med, mn = _time_launches(lambda i: kv.rope_hadamard(xk, ct, st, out=yk), 10, stream)
        byts = 2 * xk.numel() * 2 + 2 * ct.numel() * 4
        ex["rope_hadamard_bf16"] = {"ms": med, "GBps": byts / med / 1e6, "hbm_frac": byts / med / 1e6 / hbm_peak}
        del xk, yk, ct, st, ang
    return ex


def _time_graph(fns, stream, replays: int = 5, warm: bool = True):
    """Device time (ms) per launch of the launches fns[0], fns[1], ... captured back to back in ONE CUDA graph and
    replayed `replays` times (events around the replays): what a serving loop that replays a captured decode step
    sees, free of the per-launch event / host-launch overhead of `_time_launches`."""
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(stream)
    with torch.cuda.stream(side):
        if warm:            # (callers whose launches change state -- append -- pass warm = False and replay once)
            for f in fns:
                f()
        side.synchronize()
        with torch.cuda.graph(g, stream=side):
            for f in fns:
                f()
    stream.wait_stream(side)
    if warm:
        g.replay()
    torch.cuda.synchronize()
    a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(replays):
        g.replay()
    b.record(stream)
    torch.cuda.synchronize()
    return a.elapsed_time(b) / (replays * len(fns))


def stored_traffic():
    """dram bytes per launch of the two kernels, from the committed ncu --set full capture (profiles/*_traffic.csv,
    the newest round that has one)."""
    out = {}
    for name in ("r02_traffic.csv", "r01c_traffic.csv"):
        path = os.path.join(ROOT, "profiles", name)
        try:
            for line in open(path).read().splitlines()[1:]:
                k, v = line.split(",")
                out.setdefault(k, int(v))
        except Exception:
            pass
    return out


def cp_shard(n_chunks: int, rank: int, world: int):
    """Context-parallel split of a sequence's chunks over the ranks: rank r holds chunks
    [lo, hi) -- contiguous, sizes differing by at most one -- and the last rank also the residual tokens."""
    base, rem = divmod(n_chunks, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def run_cp(args, kv, W, dev, dist, rank, world):
    """--mode cp: configs[4] (2-bit) with every sequence's tokens split over the N ranks.  Per step and rank:
    kvarn_decode_attention_partial over the local share -> ONE NCCL all-gather of {m, l, o[128]} per (b, q head)
    (528 B each) -> kvarn_merge_partials.  Strong scaling: the total work is fixed, value = whole-cache bytes / time."""
    sh = W.CONFIG4
    p = kv.default_params(2)
    lo, hi = cp_shard(sh.n_chunks, rank, world)
    n_tok = (hi - lo) * G + (sh.resid if rank == world - 1 else 0)
    cache = kv.Cache(p, sh.B, sh.Hkv, max(hi - lo, 1), device=dev)
    for b0 in range(0, sh.B, 4):   # every rank draws the same sequences and keeps its slice of the tokens
        K, V = W.kv_tokens(4, sh.Hkv, sh.ctx, seed=sh.seed + b0, device=dev)
        kv.prefill(p, cache.slice(b0, b0 + 4), K[:, :, lo * G:lo * G + n_tok].contiguous(), V[:, :, lo * G:lo * G + n_tok].contiguous())
        del K, V
    q = W.queries(sh.B, sh.Hq, seed=sh.seed, device=dev)
    ws = torch.empty((max(kv.decode_workspace_bytes(p, sh.B, sh.Hq, sh.Hkv, cache.max_chunks), 16),), dtype=torch.uint8, device=dev)
    part = torch.empty((sh.B, sh.Hq, kv.PART_STRIDE), dtype=torch.float32, device=dev)
    parts = torch.empty((world,) + tuple(part.shape), dtype=torch.float32, device=dev)
    out = torch.empty((sh.B, sh.Hq, D), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        kv.decode_attention_partial(p, cache, q, part=part, ws=ws)
        if dist is not None:
            dist.all_gather_into_tensor(parts, part)
        else:
            parts[0].copy_(part)
        kv.merge_partials(parts, out=out)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(int(os.environ.get("LOCAL_RANK", "0"))) if rank == 0 else None
    if dist: dist.barrier()
    torch.cuda.synchronize()
    a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(args.steps):
        step()
    b.record(stream)
    torch.cuda.synchronize()
    if dist: dist.barrier()
    clocks = sampler.stop() if sampler else None
    ms = max_over_ranks([a.elapsed_time(b) / args.steps], dist, dev)[0]
    if rank != 0:
        return
    rb = kv.record_bytes(p)
    total = sh.B * sh.Hkv * (sh.n_chunks * 2 * rb + sh.resid * 2 * D * 2) + sh.B * sh.Hq * (D * 2 + D * 4)
    hbm_peak, peak_src = peaks()
    gbs = total / (ms * 1e-3) / 1e9
    line = {"metric": "kvarn_2bit_decode_attn_GBps", "value": gbs, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[4]: 70B-shaped long-context decode, context-parallel over the ranks",
                       "B": sh.B, "Hq": sh.Hq, "Hkv": sh.Hkv, "ctx": sh.ctx, "bits": 2, "mode": "cp",
                       "exchange": "all_gather of {m, l, o[128]} per (b, q head): %d B per rank and step" % (sh.B * sh.Hq * kv.PART_STRIDE * 4),
                       "l2": "inputs larger than L2 (2.4 GB of records per step)", "parallelism": "cp%d" % world},
            "roofline": {"kernel": "decode_kernel_w<2,8,4,2,bf16> (partial) + merge_partials_kernel", "bound": "hbm",
                         "achieved": gbs / world, "peak": hbm_peak, "unit": "GB/s per GPU", "frac": gbs / world / hbm_peak,
                         "traffic": None, "peak_source": peak_src},
            "gpu_launches": 2 * args.steps, "clocks": clocks}
    print(json.dumps(compact(line)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--impl", default="kvarn", choices=["kvarn", "reference"])
    ap.add_argument("--layers", type=int, default=8)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--extras-only", action="store_true",
                    help="run only the configs[2] / [3] / [4] measurements (profiling aid)")
    ap.add_argument("--eager-step", action="store_true",
                    help="launch the step's L decode kernels one by one instead of replaying their CUDA graph")
    ap.add_argument("--only", default="", help="with --extras-only: comma-separated extras groups to run")
    ap.add_argument("--mode", default="replicas", choices=["replicas", "cp"],
                    help="replicas (default): N independent replicas of the configs[1] step; cp: configs[4] decode with every "
                         "sequence's tokens split over the N ranks (partial -> NCCL all-gather -> LSE merge)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "kvarn" else args.warmup

    from paper_2606_03458_b200 import workloads as W
    shape = W.CONFIG1
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, shape)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the KVarN path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("NCCL_DEBUG", "VERSION")    # one line per job: which NCCL carries the collectives
        dist.init_process_group("nccl", device_id=dev)

    # libkvarn.so is built in-tree (git-ignored): local rank 0 builds it if missing or stale, the others wait
    if int(os.environ.get("LOCAL_RANK", "0")) == 0:
        from paper_2606_03458_b200 import build as _build
        _build.build()
    if dist is not None:
        dist.barrier()
    from paper_2606_03458_b200 import kvarn as kv
    hbm_peak, peak_src = peaks()
    if args.mode == "cp":
        run_cp(args, kv, W, dev, dist, rank, world)
        if dist: dist.destroy_process_group()
        return
    if args.extras_only:
        if rank == 0:
            only = set(x for x in args.only.split(",") if x)
            print(json.dumps({"extras": compact(run_extras(kv, W, dev, hbm_peak, only))}))
        return
    p = kv.default_params(shape.bits)
    rb = kv.record_bytes(p)
    L = args.layers
    BH = shape.B * shape.Hkv
    n_tiles = BH * shape.n_chunks

    # ---- synthetic inputs, resident in HBM before the timed region -----------------
    Ks, Vs, caches, qs = [], [], [], []
    for l in range(L):
        K, V = W.kv_tokens(shape.B, shape.Hkv, shape.ctx, seed=replica_seed(shape.seed, l, rank), device=dev)
        Ks.append(K.view(n_tiles, G, D)); Vs.append(V.view(n_tiles, G, D))
        qs.append(W.queries(shape.B, shape.Hq, seed=replica_seed(shape.seed, l, rank), device=dev))
        c = kv.Cache(p, shape.B, shape.Hkv, shape.n_chunks, device=dev)
        c.seq_lens.fill_(shape.ctx)
        caches.append(c)
    ws = torch.empty((max(kv.decode_workspace_bytes(p, shape.B, shape.Hq, shape.Hkv, shape.n_chunks), 16),),
                     dtype=torch.uint8, device=dev)
    out = torch.empty((shape.B, shape.Hq, D), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()

    def step(i, ev=None):
        # one layer's context quantised (write path), then the decode attention of every layer of an L-layer model
        # (read path: one launch per layer, each over its own cache -- L x 37.9 MB of records, larger than L2)
        lq = i % L
        c = caches[lq]
        if ev: ev[0].record(stream)
        kv.quantize_chunk(p, Ks[lq], Vs[lq], c.k_records.view(n_tiles, rb), c.v_records.view(n_tiles, rb))
        if ev: ev[1].record(stream)
        if dec_graphs is not None:
            dec_graphs[lq].replay()            # the same L launches, captured once (what a serving loop replays per step)
        else:
            for l in range(L):
                ld = (lq + 1 + l) % L
                kv.decode_attention(p, caches[ld], qs[ld], out=out, ws=ws)
        if ev: ev[2].record(stream)

    dec_graphs = None
    for l in range(L):   # fill every cache once (untimed) so decode always reads real records
        step(l)
    if not args.eager_step:
        # the L decode launches of a step as one CUDA graph per rotation (the layer quantised in the step is decoded
        # last, after the other L - 1 caches have gone through L2)
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        graphs = []
        for r in range(L):
            g = torch.cuda.CUDAGraph()
            side.wait_stream(stream)
            with torch.cuda.stream(side):
                with torch.cuda.graph(g, stream=side):
                    for l in range(L):
                        ld = (r + 1 + l) % L
                        kv.decode_attention(p, caches[ld], qs[ld], out=out, ws=ws, stream=side)
            stream.wait_stream(side)
            graphs.append(g)
        torch.cuda.synchronize()
        dec_graphs = graphs
    for i in range(args.warmup):
        step(i)
    torch.cuda.synchronize()

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank) if rank == 0 else None
    if dist: dist.barrier()
    torch.cuda.synchronize()
    t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
    t0.record(stream)
    for i in range(args.steps):
        step(i, evs[i])
    t1.record(stream)
    torch.cuda.synchronize()
    if dist: dist.barrier()
    total_ms = t0.elapsed_time(t1)
    q_ms = sum(e[0].elapsed_time(e[1]) for e in evs) / args.steps
    d_ms = sum(e[1].elapsed_time(e[2]) for e in evs) / args.steps / L       # per decode launch: L launches between the two events
    d1_ms, _ = _time_launches(lambda i: kv.decode_attention(p, caches[i % L], qs[i % L], out=out, ws=ws), 16, stream)  # one launch per event pair
    # the decode launch alone, back to back over the rotating caches (3 x L launches = 24 at the default, 906 MB of
    # records > L2) inside one CUDA graph: no event pair, no host launch gap (SURVEY 8(d) "Timing")
    dg_ms = _time_graph([(lambda l=l: kv.decode_attention(p, caches[l % L], qs[l % L], out=out, ws=ws)) for l in range(3 * L)], stream)
    clocks = sampler.stop() if sampler else None
    total_ms, q_ms, d_ms, dg_ms, d1_ms = max_over_ranks([total_ms, q_ms, d_ms, dg_ms, d1_ms], dist, dev)

    # ---- algorithmic bytes --------------------------------------
    dec_bytes = BH * shape.n_chunks * 2 * rb + shape.B * shape.Hq * (D * 2 + D * 4)
    q_in = 2 * n_tiles * G * D * 2
    q_bytes = q_in + 2 * n_tiles * rb
    dec_gbs = dec_bytes / (d_ms * 1e-3) / 1e9
    dec_gbs_graph = dec_bytes / (dg_ms * 1e-3) / 1e9
    q_gbs = q_bytes / (q_ms * 1e-3) / 1e9
    q_tflops = 2 * n_tiles * QUANT_FLOPS_PER_TILE / (q_ms * 1e-3) / 1e12
    tok_s = shape.B * shape.ctx / (q_ms * 1e-3)

    # ---- e2e: the same step through the host-buffer C-ABI calls --------------------------
    e2e = None
    if not args.no_e2e:
        hk = Ks[0].cpu().pin_memory(); hv = Vs[0].cpu().pin_memory()
        hq = qs[0].cpu().pin_memory()
        hout = torch.empty((shape.B, shape.Hq, D), dtype=torch.float32).pin_memory()
        dq = torch.empty_like(qs[0])
        c = caches[0]
        def e2e_step():
            kv.quantize_chunk_host(p, hk, hv, Ks[0], Vs[0], c.k_records.view(n_tiles, rb), c.v_records.view(n_tiles, rb))
            kv.decode_attention_host(p, c, hq, hout, dq, out, ws)
        n_e2e = max(3, min(args.steps, 10))
        for _ in range(2): e2e_step()
        torch.cuda.synchronize()
        if dist: dist.barrier()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n_e2e): e2e_step()
        b.record(stream)
        torch.cuda.synchronize()
        e_ms = max_over_ranks([a.elapsed_time(b) / n_e2e], dist, dev)[0]
        e2e = {"value": world * dec_bytes / (e_ms * 1e-3) / 1e9, "unit": "GB/s",
               "h2d_bytes_per_step": int(hk.numel() * 2 + hv.numel() * 2 + hq.numel() * 2),
               "d2h_bytes_per_step": int(hout.numel() * 4), "ms_per_step": e_ms,
               "tokens_per_s": world * shape.B * shape.ctx / (e_ms * 1e-3),
               "note": "kvarn_quantize_chunk_host + kvarn_decode_attention_host, pinned host buffers (PCIe-bound: 268 MB K/V upload)"}

    if rank != 0:
        if dist: dist.destroy_process_group()
        return

    cpu = None
    if not args.no_cpu_baseline:
        cpu = cpu_baseline_both(shape, rb)
        cpu["gpu_over_cpu_decode"] = dec_gbs / max(cpu["value"], 1e-12)

    extras = None
    if world == 1 and not args.no_extras:
        for t in (Ks, Vs, caches, qs):
            t.clear()
        del ws, out
        torch.cuda.empty_cache()
        extras = run_extras(kv, W, dev, hbm_peak, set())

    tr = stored_traffic()
    ex = extras or {}
    frac = lambda k: (ex.get(k) or {}).get("hbm_frac")
    # the metric's kernel is the decode kernel: its roofline is `roofline`; the other kernels' fractions ride inside it
    # (the driver's record keeps the contract keys only) and, once more, at the very end of the line
    also = {"cfg1_decode_graph_frac": dec_gbs_graph / hbm_peak, "cfg1_decode_graph_us": dg_ms * 1e3,
            "cfg1_decode_single_launch_us": d1_ms * 1e3,
            "cfg2_ctx32k_decode_frac": (ex.get("cfg2_incremental") or {}).get("decode_hbm_frac"),
            "cfg4_2bit_frac": frac("decode_cfg4_2bit"), "cfg4_4bit_frac": frac("decode_cfg4_4bit"),
            "long_g4_2bit_frac": frac("decode_long_g4_2bit"), "long_g4_4bit_frac": frac("decode_long_g4_4bit"),
            "long_g4_2bit_digits2_frac": frac("decode_long_g4_2bit_digits2"), "cfg4_2bit_digits2_frac": frac("decode_cfg4_2bit_digits2"),
            "quantize_alu_frac": q_tflops / FP32_PEAK_TFLOPS_NOMINAL, "quantize_hbm_frac": q_gbs / hbm_peak,
            "block_dense_nq32_us_per_token": (ex.get("block_dense_long_g4_2bit_nq32") or {}).get("us_per_query_token"),
            "block_dense_nq32_tensor_frac": (ex.get("block_dense_long_g4_2bit_nq32") or {}).get("tensor_frac"),
            "block_dense_nq128_us_per_token": (ex.get("block_dense_long_g4_2bit_nq128") or {}).get("us_per_query_token"),
            "block_dense_nq128_tensor_frac": (ex.get("block_dense_long_g4_2bit_nq128") or {}).get("tensor_frac"),
            "block_int_nq8_us_per_token": (ex.get("block_long_g4_2bit_nq8") or {}).get("us_per_query_token"),
            "sink128_frac": frac("decode_long_g4_2bit_sink128"),
            "target": "north_star: decode >= 0.70 of HBM on every config, quantize >= 0.60 of HBM (ALU-bound: DESIGN 6.1)"}
    rl_dec = {"kernel": "decode_kernel<2,4,2,bf16> (configs[1])", "bound": "hbm", "achieved": dec_gbs, "peak": hbm_peak,
              "unit": "GB/s", "frac": dec_gbs / hbm_peak, "traffic": tr.get("decode_kernel"),
              "algorithmic_bytes": dec_bytes, "peak_source": peak_src, "us": d_ms * 1e3,
              "timing": "CUDA events around the step's L decode launches (replayed as one CUDA graph unless --eager-step), divided by L; "
                        "also.cfg1_decode_single_launch_us: one launch per event pair; also.cfg1_decode_graph_*: 24 launches in one CUDA graph",
              "also": also}
    rl_quant = {"kernel": "quantize_kernel<2,bf16>", "bound": "alu", "achieved": q_tflops,
                "peak": FP32_PEAK_TFLOPS_NOMINAL, "unit": "TFLOP/s", "frac": q_tflops / FP32_PEAK_TFLOPS_NOMINAL,
                "traffic": tr.get("quantize_kernel"), "algorithmic_bytes": q_bytes,
                "peak_source": "derived: 148 SM x 128 fp32 lanes x 2 x 1.965 GHz (DESIGN.md)",
                "hbm_achieved_GBps": q_gbs, "hbm_frac": q_gbs / hbm_peak, "ms": q_ms}
    dn = ex.get("block_dense_long_g4_2bit_nq128") or {}
    tp, tp_src = tensor_peak()
    rl_dense = {"kernel": "block_dense_kernel<2,bf16> (packed chunks + raw windows; + merge_partials_kernel), B16 32/8 ctx 65536, n_q = 128", "bound": "tensor",
                "achieved": dn.get("TFLOPs"), "peak": tp, "unit": "TFLOP/s", "frac": dn.get("tensor_frac"), "traffic": None,
                "peak_source": tp_src, "us": dn.get("us")} if dn else None
    line = {
        "metric": "kvarn_2bit_decode_attn_GBps", "value": world * dec_gbs, "unit": "GB/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(shape, L, args.eager_step),
        "decode_us_per_step": d_ms * 1e3, "quantize_ms_per_step": q_ms,
        "quantize_tokens_per_s": world * tok_s, "quantize_tiles_per_s": world * 2 * n_tiles / (q_ms * 1e-3),
        "extras": extras, "rooflines": {"quantize": rl_quant, "block_dense": rl_dense},
        "roofline": rl_dec, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": (1 + L) * args.steps, "clocks": clocks,
        "headline": {k: v for k, v in also.items() if k != "target"} | {"cfg1_decode_frac": dec_gbs / hbm_peak, "cfg1_decode_us": d_ms * 1e3},
    }
    print(json.dumps(compact(line)))
    if dist: dist.destroy_process_group()


if __name__ == "__main__":
    main()
