"""GPU parity: kvarn_decode_attention / kvarn_prefill / kvarn_append through the
C ABI vs the oracle's plain-definition attention over the same records
(reading R17), plus properties that hold at any size."""
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


def _build_cache(kv, p, K, V, max_chunks=None, n_sink=0):
    B, Hkv, n_tok, _ = K.shape
    mc = (n_tok // 128 + 1) if max_chunks is None else max_chunks
    cache = kv.Cache(p, B, Hkv, mc, device=K.device, resid_dtype=K.dtype, n_sink=n_sink)
    kv.prefill(p, cache, K, V)
    return cache


def _oracle_unit(kv, p, cache, b, h, g, q, n_tok, sm_scale=None):
    ns, n_chunks, r = O.cache_partition(n_tok, cache.n_sink)
    kr = cache.k_records[b, h, :n_chunks].cpu().numpy()
    vr = cache.v_records[b, h, :n_chunks].cpu().numpy()
    kres = np.concatenate([P.tile_f64(cache.k_sink[b, h, :ns]), P.tile_f64(cache.k_resid[b, h, :r])])
    vres = np.concatenate([P.tile_f64(cache.v_sink[b, h, :ns]), P.tile_f64(cache.v_resid[b, h, :r])])
    qq = P.tile_f64(q[b, h * g:(h + 1) * g])
    return P.oracle_attention_from_records(kv, p, kr, vr, kres, vres, qq, sm_scale)


def _check_all_units(kv, p, cache, q, out, n_tok, units=None, sm_scale=None):
    B, Hq, _ = q.shape
    g = Hq // cache.Hkv
    out = out.to(torch.float64).cpu().numpy()
    worst = 0.0
    for b in range(B):
        for h in range(cache.Hkv):
            if units is not None and (b, h) not in units:
                continue
            ref = _oracle_unit(kv, p, cache, b, h, g, q, n_tok, sm_scale)
            worst = max(worst, P.attn_rel_err(out[b, h * g:(h + 1) * g], ref))
    assert worst <= P.ATTN_RTOL, worst
    return worst


def test_config0_single_tile_one_query(kv):
    # configs[0]: one KV head, 128 tokens, 1 query head, fp32, 2-bit
    K, V, q, _ = W.config0()
    p = kv.default_params(2)
    Kt = torch.tensor(K, device="cuda")[None, None]
    Vt = torch.tensor(V, device="cuda")[None, None]
    qt = torch.tensor(q, device="cuda")[None, None]
    cache = _build_cache(kv, p, Kt, Vt)
    assert cache.seq_lens.tolist() == [128]
    out = kv.decode_attention(p, cache, qt)
    _check_all_units(kv, p, cache, qt, out, 128)
    # end-to-end drift vs the oracle's own cache (reported, loose gate: reading R17)
    tk, tv = O.quantize_tile(K, "k"), O.quantize_tile(V, "v")
    ref = O.decode_attention(q[None].astype(np.float64), [(tk.codes, tk.s1, tk.s2, tk.z)],
                             [(tv.codes, tv.s1, tv.s2, tv.z)], np.zeros((0, 128)), np.zeros((0, 128)))
    assert P.attn_rel_err(out[0].double().cpu().numpy(), ref) < 5e-2


@pytest.mark.parametrize("bits", [2, 4])
@pytest.mark.parametrize("Hq,Hkv", [(8, 8), (16, 8), (32, 8), (64, 8), (6, 2)])
def test_gqa_shapes_with_residual(kv, bits, Hq, Hkv):
    n_tok = 128 * 5 + 77
    K, V = W.kv_tokens(2, Hkv, n_tok, seed=21 + Hq, device="cuda")
    q = W.queries(2, Hq, seed=21 + Hq, device="cuda")
    p = kv.default_params(bits)
    cache = _build_cache(kv, p, K, V)
    out = kv.decode_attention(p, cache, q)
    _check_all_units(kv, p, cache, q, out, n_tok)


@pytest.mark.parametrize("n_tok", [0, 1, 127, 128, 129, 255, 256])
def test_ragged_lengths_and_empty(kv, n_tok):
    K, V = W.kv_tokens(3, 2, max(n_tok, 1), seed=31, device="cuda")
    K, V = K[:, :, :n_tok].contiguous(), V[:, :, :n_tok].contiguous()
    q = W.queries(3, 8, seed=31, device="cuda")
    p = kv.default_params(2)
    cache = _build_cache(kv, p, K, V, max_chunks=3)
    out = kv.decode_attention(p, cache, q)
    torch.cuda.synchronize()
    if n_tok == 0:
        assert torch.all(out == 0)            # empty sequence -> zeros
    else:
        _check_all_units(kv, p, cache, q, out, n_tok)
    if 0 < n_tok < 128:
        # residual-only cache: plain SDPA over the raw bf16 tokens (library routine)
        ref = torch.nn.functional.scaled_dot_product_attention(
            q.double().view(3, 2, 4, 128), K.double(), V.double())
        assert P.attn_rel_err(out.double().cpu().numpy().reshape(3, 2, 4, 128), ref.cpu().numpy()) <= P.ATTN_RTOL


def test_mixed_lengths_in_one_batch(kv):
    # sequences of different lengths share a launch (seq_lens is per sequence)
    p = kv.default_params(2)
    lens = [300, 128, 5, 0]
    Hkv, Hq = 2, 8
    cache = kv.Cache(p, len(lens), Hkv, 3, device="cuda")
    q = W.queries(len(lens), Hq, seed=41, device="cuda")
    singles = []
    for b, n in enumerate(lens):
        K, V = W.kv_tokens(1, Hkv, max(n, 1), seed=50 + b, device="cuda")
        K, V = K[:, :, :n].contiguous(), V[:, :, :n].contiguous()
        c1 = _build_cache(kv, p, K, V, max_chunks=3)
        cache.k_records[b], cache.v_records[b] = c1.k_records[0], c1.v_records[0]
        cache.k_resid[b], cache.v_resid[b] = c1.k_resid[0], c1.v_resid[0]
        cache.seq_lens[b] = n
        singles.append(kv.decode_attention(p, c1, q[b:b + 1].contiguous()))
    out = kv.decode_attention(p, cache, q)
    for b in range(len(lens)):
        assert torch.allclose(out[b], singles[b][0], rtol=1e-5, atol=1e-6)
    for b, n in enumerate(lens[:3]):
        ref = _oracle_unit(kv, p, cache, b, 0, 4, q, n)
        assert P.attn_rel_err(out[b, :4].double().cpu().numpy(), ref) <= P.ATTN_RTOL


def test_split_count_invariance(kv):
    n_tok = 128 * 24 + 9
    K, V = W.kv_tokens(1, 2, n_tok, seed=61, device="cuda")
    q = W.queries(1, 8, seed=61, device="cuda")
    outs = []
    for s in (1, 2, 5, 24):
        p = kv.default_params(2, splits=s)
        cache = _build_cache(kv, p, K, V)
        outs.append(kv.decode_attention(p, cache, q))
    # the partials differ only by the running maximum their 18-bit fixed-point
    # probabilities refer to: an order below ATTN_RTOL
    for o in outs[1:]:
        assert (o - outs[0]).abs().max() <= 2e-4 * outs[0].abs().max()


def test_equal_logits_give_mean_of_values_and_rotation_flags(kv):
    # q = 0 -> uniform softmax -> mean over tokens of the dequantised V
    n_tok = 256
    K, V = W.kv_tokens(1, 1, n_tok, seed=71, device="cuda")
    q = torch.zeros((1, 4, 128), device="cuda", dtype=torch.bfloat16)
    for rot in (1, 0):
        p = kv.default_params(2, rotate_k=rot, rotate_v=rot)
        cache = _build_cache(kv, p, K, V)
        out = kv.decode_attention(p, cache, q)
        vt = [kv.unpack_record(p, 1, r) for r in cache.v_records[0, 0, :2].cpu().numpy()]
        Vd = np.concatenate([O.dequantize_tile(c, a.astype(np.float64), b.astype(np.float64), z.astype(np.float64),
                                               "v", rotate_on=bool(rot)) for c, a, b, z in vt])
        assert P.attn_rel_err(out[0].double().cpu().numpy(), np.tile(Vd.mean(0), (4, 1))) <= P.ATTN_RTOL
        qn = W.queries(1, 4, seed=72, device="cuda")
        _check_all_units(kv, p, cache, qn, kv.decode_attention(p, cache, qn), n_tok)


def test_bf16_output_and_custom_scale(kv):
    n_tok = 128 * 3 + 5
    K, V = W.kv_tokens(2, 2, n_tok, seed=81, device="cuda")
    q = W.queries(2, 8, seed=81, device="cuda")
    p = kv.default_params(2)
    cache = _build_cache(kv, p, K, V)
    o32 = kv.decode_attention(p, cache, q, sm_scale=0.05)
    _check_all_units(kv, p, cache, q, o32, n_tok, sm_scale=0.05)
    p.out_dtype = kv.BF16
    o16 = kv.decode_attention(p, cache, q, sm_scale=0.05)
    assert o16.dtype == torch.bfloat16 and torch.equal(o16, o32.to(torch.bfloat16))


# configs[1], [2] (full growth) and [4] at full size: tests/test_gpu_parity_full.py


def test_append_matches_prefill_bit_for_bit(kv):
    # configs[2] in miniature: grow by per-step append across two chunk
    # boundaries; records / residual / seq_lens must equal the bulk path exactly
    B, Hkv, Hq = 3, 2, 8
    start, total = 100, 100 + 300
    K, V = W.kv_tokens(B, Hkv, total, seed=91, device="cuda")
    q = W.queries(B, Hq, seed=91, device="cuda")
    p = kv.default_params(2)
    mc = total // 128 + 1
    inc = kv.Cache(p, B, Hkv, mc, device="cuda")
    kv.prefill(p, inc, K[:, :, :start].contiguous(), V[:, :, :start].contiguous())
    check_at = {127, 128, 129, 255, 256, 257, 300, total}
    for t in range(start, total):
        kv.append(p, inc, K[:, :, t].contiguous(), V[:, :, t].contiguous())
        n = t + 1
        if n in check_at:
            assert inc.seq_lens.tolist() == [n] * B
            ref = kv.Cache(p, B, Hkv, mc, device="cuda")
            kv.prefill(p, ref, K[:, :, :n].contiguous(), V[:, :, :n].contiguous())
            nc, r = n // 128, n % 128
            assert torch.equal(inc.k_records[:, :, :nc], ref.k_records[:, :, :nc])
            assert torch.equal(inc.v_records[:, :, :nc], ref.v_records[:, :, :nc])
            assert torch.equal(inc.k_resid[:, :, :r], ref.k_resid[:, :, :r])
            assert torch.equal(inc.v_resid[:, :, :r], ref.v_resid[:, :, :r])
            out = kv.decode_attention(p, inc, q)
            assert torch.equal(out, kv.decode_attention(p, ref, q))
            _check_all_units(kv, p, inc, q, out, n, units={(0, 0), (2, 1)})
    assert int(inc.ticket.abs().sum()) == 0


def test_append_capacity_guard(kv):
    # a full cache (max_chunks*128 + 127 tokens) drops further tokens, no OOB write
    p = kv.default_params(2)
    B, Hkv = 1, 1
    cache = kv.Cache(p, B, Hkv, 1, device="cuda")
    K, V = W.kv_tokens(B, Hkv, 128 + 127, seed=95, device="cuda")
    kv.prefill(p, cache, K, V)
    before = cache.k_records.clone()
    kv.append(p, cache, K[:, :, 0].contiguous(), V[:, :, 0].contiguous())      # lengths unknown to the host
    torch.cuda.synchronize()
    assert cache.seq_lens.tolist() == [255] and torch.equal(cache.k_records, before)
    assert int(cache.ticket.sum()) == 0
    assert int(cache.overflow.item()) == 1                                     # the drop is counted on the device
    with pytest.raises(kv.KvarnError, match="KVARN_CAPACITY"):                 # ... and refused when the host can tell
        kv.append(p, cache, K[:, :, 0].contiguous(), V[:, :, 0].contiguous(), max_len_hint=255)
    kv.append_block(p, cache, K[:, :, :3].contiguous(), V[:, :, :3].contiguous())
    torch.cuda.synchronize()
    assert int(cache.overflow.item()) == 2 and cache.seq_lens.tolist() == [255]


@pytest.mark.parametrize("Hq,splits", [(8, 3), (8, 5), (8, 7), (8, 8), (8, 16), (8, 21), (64, 2), (64, 3),
                                       (64, 5), (64, 6), (64, 7), (64, 8), (64, 24)])
def test_split_merge_paths_vs_oracle(kv, Hq, splits):
    # every merge route of D7: one cluster of 2..8 CTAs (DSMEM reduce-scatter by head, g = 1 and
    # g = 8 so that a rank owns 0, 1 or several heads), and several clusters through the workspace
    n_tok = 128 * 26 + 77
    K, V = W.kv_tokens(2, 8, n_tok, seed=63, device="cuda")
    q = W.queries(2, Hq, seed=63, device="cuda")
    p = kv.default_params(2, splits=splits)
    cache = _build_cache(kv, p, K, V)
    out = kv.decode_attention(p, cache, q)
    _check_all_units(kv, p, cache, q, out, n_tok, units={(0, 0), (1, 3), (1, 7)})
    assert int(cache.decode_ticket.abs().sum()) == 0
    # a second call on the same cache (tickets self-reset) gives the same bits
    assert torch.equal(out, kv.decode_attention(p, cache, q))


def test_config2_shape_incremental_decode(kv):
    # configs[2] (Qwen3-4B-shaped: B=16, 32 q / 8 KV heads) around the first append boundaries:
    # prefill 512 tokens, then append + decode per step; oracle on sampled units at the context
    # lengths SURVEY 8(d) names (639, 640, 641) -- the later growth to 32768 repeats these steps
    s = W.CONFIG2
    start, stop = 512, 642
    K, V = W.kv_tokens(s.B, s.Hkv, stop, seed=s.seed, device="cuda")
    q = W.queries(s.B, s.Hq, seed=s.seed, device="cuda")
    p = kv.default_params(2)
    cache = kv.Cache(p, s.B, s.Hkv, 8, device="cuda")
    kv.prefill(p, cache, K[:, :, :start].contiguous(), V[:, :, :start].contiguous())
    out = kv.decode_attention(p, cache, q)
    _check_all_units(kv, p, cache, q, out, start, units={(0, 0), (15, 7)})
    for t in range(start, stop):
        kv.append(p, cache, K[:, :, t].contiguous(), V[:, :, t].contiguous())
        out = kv.decode_attention(p, cache, q)
        if t + 1 in (513, 639, 640, 641):
            assert cache.seq_lens.tolist() == [t + 1] * s.B
            _check_all_units(kv, p, cache, q, out, t + 1, units={(0, 0), (7, 3), (15, 7)})


@pytest.mark.parametrize("bits,Hq,n_tok,splits", [(2, 32, 128 * 40 + 5, 0), (2, 64, 128 * 33, 6), (4, 32, 128 * 9 + 127, 0),
                                                   (2, 8, 128 * 50, 24)])
def test_decode_is_deterministic_over_repeats(kv, bits, Hq, n_tok, splits):
    # compute-sanitizer is closed on this pool, so shared-memory / DSMEM hazards are hunted by repetition:
    # the kernel has no float atomics, hence any bit that changes between identical launches is a race
    K, V = W.kv_tokens(4, 8, n_tok, seed=71, device="cuda")
    q = W.queries(4, Hq, seed=71, device="cuda")
    p = kv.default_params(bits, splits=splits)
    cache = _build_cache(kv, p, K, V)
    ref = kv.decode_attention(p, cache, q).clone()
    out = torch.empty_like(ref)
    for _ in range(200):
        kv.decode_attention(p, cache, q, out=out)
        assert torch.equal(out, ref)
    _check_all_units(kv, p, cache, q, ref, n_tok, units={(0, 0), (3, 7)})


# ---------------------------------------------------------------- FP16 sink region
@pytest.mark.parametrize("S,n_tok", [(128, 10), (128, 128), (128, 129), (128, 128 + 128 * 3 + 5), (32, 20),
                                     (32, 32 + 128 * 5), (32, 32 + 128 * 9 + 127), (64, 64 + 128 * 30 + 1)])
def test_sink_region_prefill_and_decode(kv, S, n_tok):
    K, V = W.kv_tokens(3, 8, n_tok, seed=81, device="cuda")
    q = W.queries(3, 32, seed=81, device="cuda")
    p = kv.default_params(2)
    cache = _build_cache(kv, p, K, V, n_sink=S)
    ns, nc, r = O.cache_partition(n_tok, S)
    assert cache.seq_lens.tolist() == [n_tok] * 3
    # the sink and residual regions hold the caller's raw tokens, the records the chunks after the sink
    assert torch.equal(cache.k_sink[:, :, :ns], K[:, :, :ns]) and torch.equal(cache.v_sink[:, :, :ns], V[:, :, :ns])
    assert torch.equal(cache.k_resid[:, :, :r], K[:, :, n_tok - r:]) and torch.equal(cache.v_resid[:, :, :r], V[:, :, n_tok - r:])
    if nc:
        kr, vr = kv.quantize_chunk(p, K[:, :, ns:ns + 128 * nc].reshape(-1, 128, 128).contiguous(),
                                   V[:, :, ns:ns + 128 * nc].reshape(-1, 128, 128).contiguous())
        assert torch.equal(cache.k_records[:, :, :nc].reshape(-1, cache.rb), kr)
        assert torch.equal(cache.v_records[:, :, :nc].reshape(-1, cache.rb), vr)
    out = kv.decode_attention(p, cache, q)
    _check_all_units(kv, p, cache, q, out, n_tok, units={(0, 0), (2, 7)})
    # (no end-to-end gate against the oracle's own codes here: on this peaked synthetic data a one-ulp
    # FP8 flip of a stored scale -- a legal tie, reading R17 -- moves the output by ~10 %; parity is the
    # exact comparison of the stored regions above plus attention over the GPU's own records)


@pytest.mark.parametrize("splits", [0, 3, 8, 16])
def test_sink_region_with_every_merge_route(kv, splits):
    n_tok = 128 + 128 * 20 + 77
    K, V = W.kv_tokens(2, 8, n_tok, seed=83, device="cuda")
    q = W.queries(2, 64, seed=83, device="cuda")
    p = kv.default_params(2, splits=splits)
    cache = _build_cache(kv, p, K, V, n_sink=128)
    out = kv.decode_attention(p, cache, q)
    _check_all_units(kv, p, cache, q, out, n_tok, units={(0, 0), (1, 5)})
    assert torch.equal(out, kv.decode_attention(p, cache, q))


def test_sink_region_append_matches_prefill(kv):
    # grow from inside the sink region across its end and two chunk boundaries
    B, Hkv, Hq, S = 2, 2, 8, 32
    start, total = 20, 32 + 128 * 2 + 9
    K, V = W.kv_tokens(B, Hkv, total, seed=85, device="cuda")
    q = W.queries(B, Hq, seed=85, device="cuda")
    p = kv.default_params(2)
    mc = 3
    inc = kv.Cache(p, B, Hkv, mc, device="cuda", n_sink=S)
    kv.prefill(p, inc, K[:, :, :start].contiguous(), V[:, :, :start].contiguous())
    for t in range(start, total):
        kv.append(p, inc, K[:, :, t].contiguous(), V[:, :, t].contiguous())
        n = t + 1
        if n in (31, 32, 33, 32 + 127, 32 + 128, 32 + 129, 32 + 256, total):
            assert inc.seq_lens.tolist() == [n] * B
            ref = kv.Cache(p, B, Hkv, mc, device="cuda", n_sink=S)
            kv.prefill(p, ref, K[:, :, :n].contiguous(), V[:, :, :n].contiguous())
            ns, nc, r = O.cache_partition(n, S)
            assert torch.equal(inc.k_sink[:, :, :ns], ref.k_sink[:, :, :ns]) and torch.equal(inc.v_sink[:, :, :ns], ref.v_sink[:, :, :ns])
            assert torch.equal(inc.k_records[:, :, :nc], ref.k_records[:, :, :nc])
            assert torch.equal(inc.v_records[:, :, :nc], ref.v_records[:, :, :nc])
            assert torch.equal(inc.k_resid[:, :, :r], ref.k_resid[:, :, :r]) and torch.equal(inc.v_resid[:, :, :r], ref.v_resid[:, :, :r])
            out = kv.decode_attention(p, inc, q)
            assert torch.equal(out, kv.decode_attention(p, ref, q))
            _check_all_units(kv, p, inc, q, out, n, units={(0, 0), (1, 1)})
    assert int(inc.ticket.abs().sum()) == 0


@pytest.mark.parametrize("bits,digits", [(2, 0), (2, 2), (2, 4), (4, 0), (4, 4)])
@pytest.mark.parametrize("Hq", [32, 64])
def test_decode_digit_plane_modes(kv, bits, digits, Hq):
    # kvarn_params::decode_digits: 0 = q~ 22 bits / p~ 16 bits (default), 2 = 16 / 16 (fastest), 4 = 22 / 22; every mode
    # against the oracle at the north_star tolerance, on a long-ish context (mode 2 is measured up to 1.1e-3 on
    # short peaked ones: DESIGN.md 6.2) and with a residual window
    n_tok = 128 * 40 + 19
    K, V = W.kv_tokens(2, 8, n_tok, seed=97, device="cuda")
    q = W.queries(2, Hq, seed=97, device="cuda")
    p = kv.default_params(bits, decode_digits=digits)
    cache = _build_cache(kv, p, K, V)
    out = kv.decode_attention(p, cache, q)
    worst = _check_all_units(kv, p, cache, q, out, n_tok, units={(0, 0), (1, 3), (1, 7)})
    ref4 = kv.decode_attention(kv.default_params(bits, decode_digits=4), cache, q)
    assert (out - ref4).abs().max() <= P.ATTN_RTOL * ref4.abs().max()
