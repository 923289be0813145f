"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NO KVarN arithmetic (no Hadamard, no VarN, no quantisation,
no attention): it only draws random tensors with the shapes and value
distributions DESIGN.md ("Input recipe") states.  It is the one module both the
oracle-side tests and the CUDA-side tests/bench import, so that both see the
same numbers.  It never imports the CUDA binding or the oracle.

The tensors stand in for the KV caches of the paper's Llama-3.1-8B / Qwen3-4B
workloads: same shapes (head_dim 128, 128-token chunks,
GQA 32/8 and 64/8), channel-wise outliers and a high-norm "sink" token as the
paper describes K; none of the paper's datasets or model
weights are involved.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import torch

D = 128        # head_dim
CHUNK = 128    # tokens per quantisation group (G)


@dataclass(frozen=True)
class DecodeShape:
    name: str
    B: int
    Hq: int
    Hkv: int
    ctx: int            # tokens per sequence (chunks = ctx // 128, resid = ctx % 128)
    bits: int = 2
    seed: int = 0

    @property
    def g(self) -> int:
        return self.Hq // self.Hkv

    @property
    def n_chunks(self) -> int:
        return self.ctx // CHUNK

    @property
    def resid(self) -> int:
        return self.ctx % CHUNK


CONFIG1 = DecodeShape("cfg1_llama31_8b_decode", B=8, Hq=32, Hkv=8, ctx=8192, bits=2, seed=1)
CONFIG2 = DecodeShape("cfg2_qwen3_4b_incremental", B=16, Hq=32, Hkv=8, ctx=32768, bits=2, seed=2)
CONFIG4 = DecodeShape("cfg4_70b_long_decode", B=64, Hq=64, Hkv=8, ctx=65536 + 64, bits=2, seed=4)


def config0():
    """Config 0 -- single tile, numpy seed 0 (BASELINE.json configs[0]).

    K, V fp32 [128 tok, 128 ch]; q fp32 [128].  K ~ N(0,1) with 4 outlier
    channels x20 and token 0 x10; V ~ N(0,1).
    """
    g = np.random.default_rng(0)
    K = g.standard_normal((CHUNK, D)).astype(np.float32)
    V = g.standard_normal((CHUNK, D)).astype(np.float32)
    q = g.standard_normal(D).astype(np.float32)
    oc = g.choice(D, 4, replace=False)
    K[:, oc] *= 20.0
    K[0, :] *= 10.0
    return K, V, q, np.sort(oc)


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def kv_tokens(B: int, Hkv: int, n_tok: int, seed: int, device="cpu",
              sink_first: bool = True, token_outlier_frac: float = 0.0,
              token_outlier_scale: float = 8.0, dtype=torch.bfloat16):
    """K, V of shape [B, Hkv, n_tok, 128] in ``dtype`` (configs 1-4 recipe).

    K = N(0,1) * m_c with m_c = exp(N(0,1)) per (head, channel) (log-normal
    channel magnitudes), token 0 of every sequence x10 ("sink"), optionally a
    Bernoulli(token_outlier_frac) subset of tokens x token_outlier_scale
    (config 3: 1 % x8).  V = N(0,1).
    """
    g = _gen(seed, device)
    m_c = torch.exp(torch.randn((1, Hkv, 1, D), generator=g, device=device))
    K = torch.randn((B, Hkv, n_tok, D), generator=g, device=device)
    K.mul_(m_c)
    if sink_first and n_tok > 0:
        K[:, :, 0, :] *= 10.0
    if token_outlier_frac > 0:
        mask = torch.rand((B, Hkv, n_tok, 1), generator=g, device=device) < token_outlier_frac
        K.mul_(torch.where(mask, torch.tensor(token_outlier_scale, device=device),
                           torch.tensor(1.0, device=device)))
    V = torch.randn((B, Hkv, n_tok, D), generator=g, device=device)
    return K.to(dtype), V.to(dtype)


def queries(B: int, Hq: int, seed: int, device="cpu", dtype=torch.bfloat16):
    """q ~ N(0,1), shape [B, Hq, 128]."""
    g = _gen(seed + 7919, device)
    return torch.randn((B, Hq, D), generator=g, device=device).to(dtype)


def quantizer_sweep_tiles(Hkv: int, n_tok: int, seed: int = 3, device="cpu"):
    """Config 3: K, V [Hkv, n_tok, 128] bf16 (batch 1), K with log-normal
    channel scales and 1 % token-norm outliers x8, V ~ N(0,1)."""
    K, V = kv_tokens(1, Hkv, n_tok, seed, device=device, sink_first=False,
                     token_outlier_frac=0.01, token_outlier_scale=8.0)
    return K[0], V[0]


def offset_tile(seed: int = 11, offset: float = 6.0, device="cpu"):
    """A K tile whose channels carry large offsets ("in some cases have
    large offsets"): N(0,1) + offset * N(0,1) per channel.  fp32 [128, 128]."""
    g = _gen(seed, device)
    X = torch.randn((CHUNK, D), generator=g, device=device)
    off = offset * torch.randn((1, D), generator=g, device=device)
    return (X + off).to(torch.float32)
