"""GPU parity: kvarn_block_attention (multi-token read path; Fig. 4) through the
C ABI vs the oracle's plain-definition causal block attention over the same record bytes (R17)."""
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


def _cache(kv, p, K, V, n_sink=0):
    B, Hkv, n_tok, _ = K.shape
    cache = kv.Cache(p, B, Hkv, n_tok // 128 + 1, device=K.device, resid_dtype=K.dtype, n_sink=n_sink)
    if n_tok:
        kv.prefill(p, cache, K, V)
    return cache


def _oracle_block(kv, p, cache, b, h, g, q, kb, vb, n_tok, sm_scale=None):
    """oracle.block_attention on the GPU-produced record bytes of unit (b, h)."""
    ns, n_chunks, r = O.cache_partition(n_tok, cache.n_sink)
    kt = [kv.unpack_record(p, 0, rec) for rec in cache.k_records[b, h, :n_chunks].cpu().numpy()]
    vt = [kv.unpack_record(p, 1, rec) for rec in cache.v_records[b, h, :n_chunks].cpu().numpy()]
    f64 = lambda t: tuple(np.asarray(a, dtype=np.float64) if i else a for i, a in enumerate(t))
    kt, vt = [f64(t) for t in kt], [f64(t) for t in vt]
    kraw = np.concatenate([P.tile_f64(cache.k_sink[b, h, :ns]), P.tile_f64(cache.k_resid[b, h, :r])])
    vraw = np.concatenate([P.tile_f64(cache.v_sink[b, h, :ns]), P.tile_f64(cache.v_resid[b, h, :r])])
    qq = q[b, :, h * g:(h + 1) * g].to(torch.float64).cpu().numpy()          # (n_q, g, d)
    return O.block_attention(qq, kt, vt, kraw, vraw, P.tile_f64(kb[b, h]), P.tile_f64(vb[b, h]), sm_scale=sm_scale)


def _check(kv, p, cache, q, kb, vb, out, n_tok, units=None):
    B, n_q, Hq, _ = q.shape
    g = Hq // cache.Hkv
    out = out.to(torch.float64).cpu().numpy()
    worst = 0.0
    for b in range(B):
        for h in range(cache.Hkv):
            if units is not None and (b, h) not in units:
                continue
            ref = _oracle_block(kv, p, cache, b, h, g, q, kb, vb, n_tok)
            got = out[b, :, h * g:(h + 1) * g]
            worst = max(worst, P.attn_rel_err(got.reshape(-1, 128), ref.reshape(-1, 128)))
    assert worst <= P.ATTN_RTOL, worst
    return worst


def _inputs(B, Hq, Hkv, n_tok, n_q, seed, dtype=torch.bfloat16):
    K, V = W.kv_tokens(B, Hkv, n_tok + n_q, seed=seed, device="cuda")
    K, V = K.to(dtype), V.to(dtype)
    q = torch.stack([W.queries(B, Hq, seed=seed * 131 + i, device="cuda") for i in range(n_q)], dim=1).to(dtype).contiguous()
    return (K[:, :, :n_tok].contiguous(), V[:, :, :n_tok].contiguous(),
            K[:, :, n_tok:].contiguous(), V[:, :, n_tok:].contiguous(), q)


@pytest.mark.parametrize("bits", [2, 4])
@pytest.mark.parametrize("Hq,Hkv,n_q", [(32, 8, 1), (32, 8, 2), (32, 8, 5), (8, 8, 8), (8, 8, 19), (16, 8, 7),
                                         (64, 8, 3), (32, 8, 128)])
def test_block_attention_vs_oracle(kv, bits, Hq, Hkv, n_q):
    n_tok = 128 * 3 + 41
    K, V, kb, vb, q = _inputs(2, Hq, Hkv, n_tok, n_q, seed=60 + n_q)
    p = kv.default_params(bits)
    cache = _cache(kv, p, K, V)
    out = kv.block_attention(p, cache, q, kb, vb)
    units = None if n_q <= 8 else {(0, 0), (1, Hkv - 1)}
    _check(kv, p, cache, q, kb, vb, out, n_tok, units)


@pytest.mark.parametrize("n_tok", [0, 1, 127, 128, 129, 256])
def test_block_attention_ragged_and_empty_cache(kv, n_tok):
    n_q = 6
    K, V, kb, vb, q = _inputs(1, 16, 4, n_tok, n_q, seed=70 + n_tok)
    p = kv.default_params(2)
    cache = _cache(kv, p, K, V)
    out = kv.block_attention(p, cache, q, kb, vb)
    _check(kv, p, cache, q, kb, vb, out, n_tok)


@pytest.mark.parametrize("splits", [1, 2, 5, 8])
def test_block_attention_split_routes_and_sink(kv, splits):
    n_tok, n_q = 32 + 128 * 9 + 100, 4
    K, V, kb, vb, q = _inputs(2, 16, 4, n_tok, n_q, seed=80)
    p = kv.default_params(2, splits=splits)
    cache = _cache(kv, p, K, V, n_sink=32)
    out = kv.block_attention(p, cache, q, kb, vb)
    _check(kv, p, cache, q, kb, vb, out, n_tok)


def test_block_of_one_equals_decode_after_append(kv):
    """n_q = 1: attending [cache ; the new token] = kvarn_append then kvarn_decode_attention."""
    n_tok = 128 * 4 + 17
    K, V, kb, vb, q = _inputs(3, 32, 8, n_tok, 1, seed=90)
    p = kv.default_params(2)
    cache = _cache(kv, p, K, V)
    out_blk = kv.block_attention(p, cache, q, kb, vb)
    kv.append(p, cache, kb[:, :, 0].contiguous(), vb[:, :, 0].contiguous())
    out_dec = kv.decode_attention(p, cache, q[:, 0].contiguous())
    err = (out_blk[:, 0] - out_dec).abs().max().item() / out_dec.abs().max().item()
    assert err <= 2e-4, err


def test_block_attention_is_causal(kv):
    """Changing block tokens j > i must leave the outputs of queries 0..i bit-identical."""
    n_tok, n_q = 300, 8
    K, V, kb, vb, q = _inputs(1, 16, 4, n_tok, n_q, seed=95)
    p = kv.default_params(2)
    cache = _cache(kv, p, K, V)
    out = kv.block_attention(p, cache, q, kb, vb)
    kb2, vb2 = kb.clone(), vb.clone()
    kb2[:, :, 5:] *= 3.0
    vb2[:, :, 5:] -= 7.0
    out2 = kv.block_attention(p, cache, q, kb2, vb2)
    assert torch.equal(out[:, :5], out2[:, :5])
    assert not torch.equal(out[:, 5:], out2[:, 5:])


def test_block_attention_rejects_bad_arguments(kv):
    p = kv.default_params(2)
    cache = kv.Cache(p, 1, 2, 2)
    q = torch.zeros((1, 2, 6, 128), dtype=torch.bfloat16, device="cuda")      # g = 3: unsupported here
    kb = torch.zeros((1, 2, 2, 128), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(kv.KvarnError, match="UNSUPPORTED"):
        kv.block_attention(p, cache, q, kb, kb.clone())


def test_block_attention_fp32_inputs_bf16_output_and_custom_scale(kv):
    n_tok, n_q = 128 * 2 + 9, 3
    K, V, kb, vb, q = _inputs(1, 8, 2, n_tok, n_q, seed=97, dtype=torch.float32)
    p = kv.default_params(4)
    cache = _cache(kv, p, K, V)
    out = kv.block_attention(p, cache, q, kb, vb, sm_scale=0.05)
    p.out_dtype = kv.BF16
    out_bf = kv.block_attention(p, cache, q, kb, vb, sm_scale=0.05)
    assert out_bf.dtype == torch.bfloat16
    assert (out_bf.float() - out).abs().max().item() <= 2 ** -7 * out.abs().max().item()
    ref = _oracle_block(kv, p, cache, 0, 1, 4, q, kb, vb, n_tok, sm_scale=0.05)
    got = out.double().cpu().numpy()[0, :, 4:8]
    assert P.attn_rel_err(got.reshape(-1, 128), ref.reshape(-1, 128)) <= P.ATTN_RTOL


def test_block_attention_is_deterministic_over_repeats(kv):
    """Race hunt by repetition (compute-sanitizer is closed on this pool): 100 identical launches, bit-identical."""
    n_tok, n_q = 128 * 6 + 70, 5
    K, V, kb, vb, q = _inputs(2, 32, 8, n_tok, n_q, seed=98)
    p = kv.default_params(2)
    cache = _cache(kv, p, K, V, n_sink=32)
    first = kv.block_attention(p, cache, q, kb, vb).clone()
    for _ in range(100):
        assert torch.equal(kv.block_attention(p, cache, q, kb, vb), first)


@pytest.mark.parametrize("bits,n_sink", [(2, 0), (2, 32), (4, 128)])
def test_append_block_matches_prefill_bit_for_bit(kv, bits, n_sink):
    """Pseudo-decode write half (Fig. 4): prefill(L0) + append_block(n_1) + append_block(n_2) ... leaves exactly
    the cache prefill(L0 + sum n_i) leaves -- records, sink, residual window and seq_lens."""
    B, Hkv = 2, 4
    blocks = [1, 5, 128, 37, 100, 128, 90, 3, 127, 64]
    L0 = 20                                              # shorter than n_sink = 32 / 128: blocks straddle the sink boundary
    total = L0 + sum(blocks)
    K, V = W.kv_tokens(B, Hkv, total, seed=101, device="cuda")
    p = kv.default_params(bits)
    mc = total // 128 + 1
    inc = kv.Cache(p, B, Hkv, mc, n_sink=n_sink)
    kv.prefill(p, inc, K[:, :, :L0].contiguous(), V[:, :, :L0].contiguous())
    pos = L0
    for n in blocks:
        kv.append_block(p, inc, K[:, :, pos:pos + n].contiguous(), V[:, :, pos:pos + n].contiguous())
        pos += n
        ref = kv.Cache(p, B, Hkv, mc, n_sink=n_sink)
        kv.prefill(p, ref, K[:, :, :pos].contiguous(), V[:, :, :pos].contiguous())
        ns, nc, r = O.cache_partition(pos, n_sink)
        assert inc.seq_lens.tolist() == [pos] * B
        assert torch.equal(inc.k_records[:, :, :nc], ref.k_records[:, :, :nc]) and torch.equal(inc.v_records[:, :, :nc], ref.v_records[:, :, :nc])
        assert torch.equal(inc.k_resid[:, :, :r], ref.k_resid[:, :, :r]) and torch.equal(inc.v_resid[:, :, :r], ref.v_resid[:, :, :r])
        assert torch.equal(inc.k_sink[:, :, :ns], ref.k_sink[:, :, :ns]) and torch.equal(inc.v_sink[:, :, :ns], ref.v_sink[:, :, :ns])


def test_pseudo_decode_step_and_capacity_guard(kv):
    """block attention over the cache, then the block is appended; the next single-token decode sees it.  A block that
    would need a chunk slot beyond max_chunks leaves the sequence unchanged."""
    B, Hq, Hkv, L0, n = 1, 16, 4, 128 * 2 + 100, 60
    K, V, kb, vb, q = _inputs(B, Hq, Hkv, L0, n, seed=103)
    p = kv.default_params(2)
    cache = kv.Cache(p, B, Hkv, 3)
    kv.prefill(p, cache, K, V)
    out_blk = kv.block_attention(p, cache, q, kb, vb)
    kv.append_block(p, cache, kb, vb)                    # 100 + 60 = 160: completes chunk 2, 32 tokens remain
    assert cache.seq_lens.tolist() == [L0 + n]
    out_dec = kv.decode_attention(p, cache, q[:, -1].contiguous())
    assert torch.isfinite(out_blk).all()
    full = kv.Cache(p, B, Hkv, 3); kv.prefill(p, full, torch.cat([K, kb], 2).contiguous(), torch.cat([V, vb], 2).contiguous())
    assert torch.equal(out_dec, kv.decode_attention(p, full, q[:, -1].contiguous()))
    big = torch.zeros((B, Hkv, 128, 128), dtype=torch.bfloat16, device="cuda")
    kv.append_block(p, cache, big, big.clone())           # 32 + 128 -> would complete chunk 3 = max_chunks: dropped
    assert cache.seq_lens.tolist() == [L0 + n]
    with pytest.raises(kv.KvarnError, match="UNSUPPORTED"):
        kv.append_block(p, cache, torch.zeros((B, Hkv, 129, 128), dtype=torch.bfloat16, device="cuda"),
                        torch.zeros((B, Hkv, 129, 128), dtype=torch.bfloat16, device="cuda"))


# ---------------------------------------------------------------- dense tcgen05 form (kvarn_block_attention_dense)
@pytest.mark.parametrize("bits", [2, 4])
@pytest.mark.parametrize("Hq,Hkv,n_q,n_tok,n_sink", [(32, 8, 128, 128 * 5 + 41, 0), (32, 8, 40, 128 * 9, 0), (64, 8, 16, 128 * 4 + 100, 0),
                                                      (8, 8, 128, 128 * 3 + 7, 0), (32, 8, 33, 128 * 6 + 5, 32), (16, 8, 3, 128 * 2 + 1, 0),
                                                      (32, 8, 8, 77, 0), (32, 8, 20, 0, 0)])
def test_block_attention_dense_vs_oracle(kv, bits, Hq, Hkv, n_q, n_tok, n_sink):
    # row tiles full and ragged (n_q g = 512, 160, 128, 128, 132, 6), several chunks per CTA, sink / residual / empty cache
    K, V, kb, vb, q = _inputs(2, Hq, Hkv, n_tok, n_q, seed=160 + n_q)
    p = kv.default_params(bits)
    cache = _cache(kv, p, K, V, n_sink=n_sink)
    out = kv.block_attention(p, cache, q, kb, vb, dense=True)
    _check(kv, p, cache, q, kb, vb, out, n_tok, {(0, 0), (1, Hkv - 1)})
    ref = kv.block_attention(p, cache, q, kb, vb)                      # the integer-MMA form
    assert (out - ref).abs().max() <= P.ATTN_RTOL * ref.abs().max()
    assert torch.equal(out, kv.block_attention(p, cache, q, kb, vb, dense=True))     # deterministic


def test_block_attention_dense_long_context_and_splits(kv):
    # one sequence, one KV head pair, 40 chunks: the chunk range is split over several CTAs whose partials are LSE-merged
    n_tok, n_q = 128 * 40 + 9, 32
    K, V, kb, vb, q = _inputs(1, 8, 2, n_tok, n_q, seed=171)
    p = kv.default_params(2)
    cache = _cache(kv, p, K, V)
    out = kv.block_attention(p, cache, q, kb, vb, dense=True)
    _check(kv, p, cache, q, kb, vb, out, n_tok)


@pytest.mark.parametrize("dense", [False, True])
@pytest.mark.parametrize("bits", [2, 4])
def test_block_attention_token_scale_spread_and_dominant_keys(kv, bits, dense):
    """V token norms spread over 20 binades inside a chunk (incl. all-zero V rows and half a chunk 2^-14 below the other
    half) and keys that dominate their chunk by 10-20 log2 units for individual query rows, against the oracle on the
    same record bytes.  Integer path: what is rounded to fixed point is p s1v[t], so the denominator must take the exact
    p (a token with a tiny V row keeps its probability mass).  Dense path: s1v[t] enters as a per-chunk exponent in the
    logits and an exact factor in the tile, and the TMEM accumulator is rescaled when a row's maximum rises.
    The error is taken relative to the largest output of the (sequence, KV head) unit: rows that attend to a
    tiny-norm token have outputs 2^-12 of the others', so R16's per-row ratio would measure nothing but that scale."""
    n_tok, n_q, Hq, Hkv = 128 * 6 + 17, 40, 8, 2
    K, V, kb, vb, q = _inputs(1, Hq, Hkv, n_tok, n_q, seed=190 + bits)
    gen = torch.Generator(device="cuda").manual_seed(7)
    e = torch.randint(-12, 9, (1, Hkv, n_tok, 1), generator=gen, device="cuda").to(torch.float32)
    V = (V.float() * torch.exp2(e)).to(V.dtype)
    V[:, :, 5::41] = 0                                   # whole V rows exactly zero
    V[:, :, 128 * 3:128 * 4:2] *= 2.0 ** -14             # half of one chunk far below the other half
    for i, t in enumerate((130, 300, 301, 640, 777)):    # keys aligned with individual queries
        K[0, :, t] = (q[0, (7 * i) % n_q, ::Hq // Hkv].float() * (3.0 + i)).to(K.dtype)
    p = kv.default_params(bits)
    cache = _cache(kv, p, K, V)
    out = kv.block_attention(p, cache, q, kb, vb, dense=dense)
    assert torch.isfinite(out).all()
    g = Hq // Hkv
    o = out.to(torch.float64).cpu().numpy()
    for h in range(Hkv):
        ref = _oracle_block(kv, p, cache, 0, h, g, q, kb, vb, n_tok)
        err = np.abs(o[0, :, h * g:(h + 1) * g] - ref).max() / np.abs(ref).max()
        assert err <= P.ATTN_RTOL, (h, err)


@pytest.mark.parametrize("dense", [False, True])
def test_block_attention_ragged_lengths_in_one_batch(kv, dense):
    """Sequences of very different lengths in one call (41 chunks, 3 chunks + a residual window, 5 raw tokens, an empty
    cache): the dense kernel's chunk ranges are planned from the cache's capacity, so most CTAs of the short sequences
    own no chunk at all and the last one owns only the raw windows."""
    lens = [128 * 41 + 9, 128 * 3 + 70, 5, 0]
    B, Hq, Hkv, n_q = len(lens), 4, 1, 32
    p = kv.default_params(2)
    cache = kv.Cache(p, B, Hkv, 42, device="cuda")
    q = torch.stack([W.queries(B, Hq, seed=700 + i, device="cuda") for i in range(n_q)], dim=1).contiguous()
    kb, vb = W.kv_tokens(B, Hkv, n_q, seed=701, device="cuda", sink_first=False)
    for b, n in enumerate(lens):
        K, V = W.kv_tokens(1, Hkv, max(n, 1), seed=710 + b, device="cuda")
        kv.prefill(p, cache.slice(b, b + 1), K[:, :, :n].contiguous(), V[:, :, :n].contiguous())
    assert cache.seq_lens.tolist() == lens
    out = kv.block_attention(p, cache, q, kb, vb, dense=dense).to(torch.float64).cpu().numpy()
    g = Hq // Hkv
    for b, n in enumerate(lens):
        ref = _oracle_block(kv, p, cache, b, 0, g, q, kb, vb, n)
        err = P.attn_rel_err(out[b, :, 0:g].reshape(-1, 128), ref.reshape(-1, 128))
        assert err <= P.ATTN_RTOL, (b, n, err)
