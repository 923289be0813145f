"""GPU parity: kvarn_decode_attention_partial + kvarn_merge_partials (context-parallel building block,
SURVEY 8(e)): a sequence split over several caches, partials merged, vs the oracle and vs the one-cache decode."""
import numpy as np
import pytest
import torch

from oracle import kvarn_oracle as O
from paper_2606_03458_b200 import workloads as W
import kvarn_parity as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def kv():
    from paper_2606_03458_b200 import kvarn
    return kvarn


def _shard_caches(kv, p, K, V, cuts):
    """caches over token ranges [cuts[i], cuts[i+1]) of every sequence (cuts at multiples of 128 except the last)."""
    caches = []
    for a, b in zip(cuts[:-1], cuts[1:]):
        c = kv.Cache(p, K.shape[0], K.shape[1], (b - a) // 128 + 1, device=K.device, resid_dtype=K.dtype)
        if b > a:
            kv.prefill(p, c, K[:, :, a:b].contiguous(), V[:, :, a:b].contiguous())
        caches.append(c)
    return caches


@pytest.mark.parametrize("bits,Hq,Hkv,splits", [(2, 32, 8, 0), (4, 16, 8, 0), (2, 64, 8, 24), (2, 8, 8, 1)])
def test_partials_merge_to_the_full_attention(kv, bits, Hq, Hkv, splits):
    B, n_tok = 2, 128 * 11 + 60
    K, V = W.kv_tokens(B, Hkv, n_tok, seed=71, device="cuda")
    q = W.queries(B, Hq, seed=71, device="cuda")
    p = kv.default_params(bits, splits=splits)
    cuts = [0, 128 * 3, 128 * 3, 128 * 8, n_tok]            # 4 "ranks", one of them empty
    caches = _shard_caches(kv, p, K, V, cuts)
    parts = torch.stack([kv.decode_attention_partial(p, c, q) for c in caches])
    assert torch.isinf(parts[1, :, :, 0]).all() and (parts[1, :, :, 1] == 0).all()      # empty share: m = -inf, l = 0
    out = kv.merge_partials(parts)
    # (1) vs the one-cache decode of the same records (chunk boundaries coincide, so the records are identical)
    full = kv.Cache(p, B, Hkv, n_tok // 128 + 1); kv.prefill(p, full, K, V)
    ref_gpu = kv.decode_attention(p, full, q)
    err = ((out - ref_gpu).abs().amax(dim=-1) / ref_gpu.abs().amax(dim=-1)).max().item()
    assert err <= 2e-4, err
    # (2) vs the oracle on the GPU's records
    g = Hq // Hkv
    o64 = out.double().cpu().numpy()
    for b, h in ((0, 0), (1, Hkv - 1)):
        ns, n_chunks, r = O.cache_partition(n_tok)
        ref = P.oracle_attention_from_records(kv, p, full.k_records[b, h, :n_chunks].cpu().numpy(),
                                              full.v_records[b, h, :n_chunks].cpu().numpy(),
                                              P.tile_f64(full.k_resid[b, h, :r]), P.tile_f64(full.v_resid[b, h, :r]),
                                              P.tile_f64(q[b, h * g:(h + 1) * g]))
        assert P.attn_rel_err(o64[b, h * g:(h + 1) * g], ref) <= P.ATTN_RTOL
    # (3) the partial's own definition: l and o of one share against the oracle's un-normalised sums
    b, h = 0, 1
    kt = [kv.unpack_record(p, 0, rec) for rec in caches[0].k_records[b, h, :3].cpu().numpy()]
    vt = [kv.unpack_record(p, 1, rec) for rec in caches[0].v_records[b, h, :3].cpu().numpy()]
    f64 = lambda t: tuple(np.asarray(a, dtype=np.float64) if i else a for i, a in enumerate(t))
    Kd = np.concatenate([O.dequantize_tile(*f64(t), kind="k") for t in kt]); Vd = np.concatenate([O.dequantize_tile(*f64(t), kind="v") for t in vt])
    logits = (P.tile_f64(q[b, h * g]) @ Kd.T) / np.sqrt(128.0) * np.log2(np.e)
    m = logits.max(); w = 2.0 ** (logits - m)
    got = parts[0, b, h * g].double().cpu().numpy()
    # m is a reference exponent (the kernel's running maximum includes the folded V scale), l and o are relative to it
    sc = 2.0 ** (got[0] - m)
    assert got[0] >= m - 60 and abs(got[1] * sc / w.sum() - 1) <= 1e-3
    assert np.abs(got[4:] * sc - w @ Vd).max() <= 2e-3 * np.abs(w @ Vd).max()


def test_merge_of_all_empty_parts_is_zero_and_bf16_out(kv):
    parts = torch.zeros((3, 2, 4, 132), dtype=torch.float32, device="cuda")
    parts[..., 0] = float("-inf")
    assert (kv.merge_partials(parts) == 0).all()
    parts[1, :, :, 0] = 0.5; parts[1, :, :, 1] = 2.0; parts[1, :, :, 4:] = 3.0
    out = kv.merge_partials(parts, out_dtype=torch.bfloat16)
    assert out.dtype == torch.bfloat16 and torch.allclose(out.float(), torch.full_like(out, 1.5, dtype=torch.float32))


def test_context_parallel_decode_helper_world_size_1(kv):
    """The torch.distributed helper (partial -> all_gather_into_tensor over NCCL -> merge) with a one-rank group
    equals the plain decode; more ranks need more GPUs than this box has."""
    import os
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29531")
    created = not dist.is_initialized()
    if created:
        dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        K, V = W.kv_tokens(2, 4, 128 * 5 + 33, seed=72, device="cuda")
        q = W.queries(2, 16, seed=72, device="cuda")
        p = kv.default_params(2)
        cache = kv.Cache(p, 2, 4, 6); kv.prefill(p, cache, K, V)
        out = kv.context_parallel_decode(p, cache, q)
        ref = kv.decode_attention(p, cache, q)
        assert (out - ref).abs().max().item() <= 2e-5 * ref.abs().max().item()
    finally:
        if created:
            dist.destroy_process_group()
