"""GPU parity at BASELINE.json's full sizes, with the sample sizes SURVEY 8(d) asks for (full for configs 0-1,
>= 1 % of the independent units for configs 2-4), the adversarial inputs of VERDICT round 1 (fixed-point
probabilities under a dominant token, channel offsets >> std) and the measured rate of storage-rounding ties.
The oracle is fanned out over the host cores (oracle/fanout.py); everything goes through the C ABI."""
import numpy as np
import pytest
import torch

from oracle import fanout
from oracle import kvarn_oracle as O
from paper_2606_03458_b200 import workloads as W
import kvarn_parity as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def kv():
    from paper_2606_03458_b200 import kvarn
    return kvarn


def _unit_job(kv, p, cache, q, b, h, g, n_tok, sm_scale=None):
    """fanout 'decode' job of unit (b, h): the GPU's own record bytes (reading R17) + raw sink / residual tokens."""
    ns, nc, r = O.cache_partition(n_tok, cache.n_sink)
    kt = [kv.unpack_record(p, 0, rec) for rec in cache.k_records[b, h, :nc].cpu().numpy()]
    vt = [kv.unpack_record(p, 1, rec) for rec in cache.v_records[b, h, :nc].cpu().numpy()]
    kraw = np.concatenate([P.tile_f64(cache.k_sink[b, h, :ns]), P.tile_f64(cache.k_resid[b, h, :r])])
    vraw = np.concatenate([P.tile_f64(cache.v_sink[b, h, :ns]), P.tile_f64(cache.v_resid[b, h, :r])])
    return (P.tile_f64(q[b, h * g:(h + 1) * g]), kt, vt, kraw, vraw, sm_scale, bool(p.rotate_k), bool(p.rotate_v))


def _check_units(kv, p, cache, q, out, n_tok, units):
    g = q.shape[1] // cache.Hkv
    refs = fanout.pmap("decode", [_unit_job(kv, p, cache, q, b, h, g, n_tok) for b, h in units])
    o = out.to(torch.float64).cpu().numpy()
    errs = [P.attn_rel_err(o[b, h * g:(h + 1) * g], ref) for (b, h), ref in zip(units, refs)]
    assert max(errs) <= P.ATTN_RTOL, (max(errs), units[int(np.argmax(errs))])
    return errs


def _check_tiles(kv, p, Kt, Vt, idx, stats):
    """Quantise the tiles idx of Kt / Vt ([n, 128, 128] on the GPU) with debug outputs and compare each with the oracle."""
    ii = torch.as_tensor(idx, device=Kt.device)
    Ks, Vs = Kt[ii].contiguous(), Vt[ii].contiguous()
    kr, vr, dbg = kv.quantize_chunk(p, Ks, Vs, debug=True)
    torch.cuda.synchronize()
    kb, imb, aux = dbg.k_best.cpu().numpy(), dbg.imb.cpu().numpy(), dbg.aux.cpu().numpy()
    for kind, (X, R) in enumerate(((Ks, kr), (Vs, vr))):
        Xs = X.to(torch.float32).cpu().numpy()
        P.check_quantized_tiles(kv, p, kind, list(Xs), list(R.cpu().numpy()), kb[kind], imb[kind], aux[kind], stats)
    return kr, vr


# ------------------------------------------------------------------------------------------------ configs[1]
def test_config1_full_every_unit_and_quantizer_sample(kv):
    """configs[1] (B=8, 32 q / 8 KV heads, ctx 8192, bf16, x10 sink token), in the launch configuration bench.py
    times: attention of ALL 64 (sequence, KV head) units vs the oracle; quantizer records of 128 of the 8192 tiles
    per kind (1.6 %: tile 0 of every unit -- the one with the sink token -- plus 64 seeded others) vs the oracle;
    end to end on 4 units (printed; reading R17): the GPU's output against attention over the oracle's OWN cache
    and against attention over the raw K, V.  The two caches hold the same codes but -- Alg. 1 line 18 being
    degenerate (R10) -- often a different iterate's scales, whose FP8 roundings differ; on this peaked synthetic
    data (logits up to +-57) that moves single outputs by ~10 %.  What is gated is that the GPU's cache is as good
    a quantisation as the oracle's: its error against the un-quantised attention is not larger."""
    s = W.CONFIG1
    K, V = W.kv_tokens(s.B, s.Hkv, s.ctx, seed=s.seed, device="cuda")
    q = W.queries(s.B, s.Hq, seed=s.seed, device="cuda")
    p = kv.default_params(2)
    cache = kv.Cache(p, s.B, s.Hkv, s.n_chunks, device="cuda")
    kv.prefill(p, cache, K, V)
    out = kv.decode_attention(p, cache, q)
    units = [(b, h) for b in range(s.B) for h in range(s.Hkv)]
    errs = _check_units(kv, p, cache, q, out, s.ctx, units)
    n_tiles = s.B * s.Hkv * s.n_chunks
    Kt, Vt = K.view(n_tiles, 128, 128), V.view(n_tiles, 128, 128)
    rng = np.random.default_rng(1)
    idx = sorted(set(range(0, n_tiles, s.n_chunks)) | set(rng.choice(n_tiles, 64, replace=False).tolist()))
    stats = {}
    kr, vr = _check_tiles(kv, p, Kt, Vt, idx, stats)
    P.assert_mismatch_budget(stats)
    # the sampled launch and the full prefill launch write the same bytes
    ii = torch.as_tensor(idx, device="cuda")
    assert torch.equal(cache.k_records.view(n_tiles, -1)[ii], kr) and torch.equal(cache.v_records.view(n_tiles, -1)[ii], vr)
    du = [(0, 0), (2, 5), (5, 1), (7, 7)]
    own = fanout.pmap("cache_attention", [(P.tile_f64(q[b, h * s.g:(h + 1) * s.g]), P.tile_f64(K[b, h]), P.tile_f64(V[b, h]), 0, 2)
                                          for b, h in du])
    o = out.double().cpu().numpy()
    drift = [P.attn_rel_err(o[b, h * s.g:(h + 1) * s.g], ref[0]) for (b, h), ref in zip(du, own)]
    e_gpu = [P.attn_rel_err(o[b, h * s.g:(h + 1) * s.g], ref[1]) for (b, h), ref in zip(du, own)]
    e_orc = [P.attn_rel_err(ref[0], ref[1]) for ref in own]
    print(f"configs[1]: attention vs oracle over the GPU's records: max {max(errs):.2e} over {len(units)} units; "
          f"end to end: drift vs the oracle's own cache {['%.1e' % d for d in drift]}, error vs un-quantised attention "
          f"GPU cache {['%.1e' % d for d in e_gpu]} / oracle cache {['%.1e' % d for d in e_orc]}; quantizer {stats}")
    assert np.mean(e_gpu) <= 1.5 * np.mean(e_orc) + 1e-3 and max(drift) <= 0.5


# ------------------------------------------------------------------------------------------------ configs[2]
def test_config2_full_growth_512_to_32768(kv):
    """configs[2] (B=16, 32 q / 8 KV heads): prefill 512 tokens, then ONE kvarn_append + ONE kvarn_decode_attention
    per step up to 32 768 tokens (32 256 steps, 252 chunk boundaries).  At the end every record, the residual window
    and seq_lens equal a bulk prefill of the whole sequence bit for bit; oracle attention on 3 of the 128 units
    (2.3 %) at ctx 4096, 32 767 and 32 768."""
    s = W.CONFIG2
    start = 512
    K, V = W.kv_tokens(s.B, s.Hkv, s.ctx, seed=s.seed, device="cuda")
    q = W.queries(s.B, s.Hq, seed=s.seed, device="cuda")
    p = kv.default_params(2)
    inc = kv.Cache(p, s.B, s.Hkv, s.n_chunks, device="cuda")
    kv.prefill(p, inc, K[:, :, :start].contiguous(), V[:, :, :start].contiguous())
    Kt = K.permute(2, 0, 1, 3).contiguous()      # [ctx][B][Hkv][128]: one contiguous token per step
    Vt = V.permute(2, 0, 1, 3).contiguous()
    ws = torch.empty((max(kv.decode_workspace_bytes(p, s.B, s.Hq, s.Hkv, s.n_chunks), 16),), dtype=torch.uint8, device="cuda")
    out = torch.empty((s.B, s.Hq, 128), dtype=torch.float32, device="cuda")
    units = [(0, 0), (9, 3), (15, 7)]
    worst = {}
    for t in range(start, s.ctx):
        kv.append(p, inc, Kt[t], Vt[t], max_len_hint=t)
        kv.decode_attention(p, inc, q, out=out, ws=ws)
        n = t + 1
        if n in (4096, s.ctx - 1, s.ctx):
            assert inc.seq_lens.tolist() == [n] * s.B
            worst[n] = max(_check_units(kv, p, inc, q, out, n, units))
    assert int(inc.overflow.item()) == 0 and int(inc.ticket.abs().sum()) == 0
    ref = kv.Cache(p, s.B, s.Hkv, s.n_chunks, device="cuda")
    kv.prefill(p, ref, K, V)
    assert torch.equal(inc.k_records, ref.k_records) and torch.equal(inc.v_records, ref.v_records)
    assert torch.equal(inc.seq_lens, ref.seq_lens)
    assert torch.equal(out, kv.decode_attention(p, ref, q))
    print(f"configs[2]: attention vs oracle at ctx {sorted(worst)}: {['%.2e' % worst[k] for k in sorted(worst)]}")


# ------------------------------------------------------------------------------------------------ configs[3]
@pytest.mark.parametrize("bits", [2, 4])
def test_config3_full_size_one_percent_of_tiles(kv, bits):
    """configs[3] at full size: 8 KV heads x 2^20 tokens = 131 072 K + 131 072 V tiles in ONE launch (the launch
    bench.py's extras time).  1 312 seeded tiles per kind (1.0 %) are compared with the oracle element by element
    (their records taken from the big launch), the rest by properties that hold at any size."""
    n_tok = 1 << 20
    K, V = W.quantizer_sweep_tiles(8, n_tok, seed=3, device="cuda")
    n_tiles = 8 * n_tok // 128
    Kt, Vt = K.view(n_tiles, 128, 128), V.view(n_tiles, 128, 128)
    p = kv.default_params(bits)
    k_rec, v_rec = kv.quantize_chunk(p, Kt, Vt)
    rng = np.random.default_rng(3)
    idx = sorted(set([0, 1, n_tiles // 2, n_tiles - 2, n_tiles - 1]) | set(rng.choice(n_tiles, 1307, replace=False).tolist()))
    assert len(idx) >= 1311
    stats = {}
    kr, vr = _check_tiles(kv, p, Kt, Vt, idx, stats)
    P.assert_mismatch_budget(stats)
    ii = torch.as_tensor(idx, device="cuda")
    assert torch.equal(k_rec[ii], kr) and torch.equal(v_rec[ii], vr)      # the big launch wrote the same bytes
    assert bool((k_rec[:, :64].any(dim=1)).all()) and bool((v_rec[:, :64].any(dim=1)).all())   # no record is empty
    print(f"configs[3] {bits}-bit: {stats}")


# ------------------------------------------------------------------------------------------------ configs[4]
@pytest.mark.parametrize("bits", [2, 4])
def test_config4_full_size_eight_units(kv, bits):
    """configs[4] at full size (B=64, 64 q / 8 KV heads, ctx 65 536 + 64-token bf16 residual), in the launch
    configuration bench.py's extras time; oracle attention on 8 of the 512 units (1.6 %); end-to-end drift vs the
    oracle's own cache and vs un-quantised attention on one unit (512 chunks re-quantised by the oracle), printed."""
    s = W.CONFIG4
    p = kv.default_params(bits)
    cache = kv.Cache(p, s.B, s.Hkv, s.n_chunks, device="cuda")
    keep = {}
    for b0 in range(0, s.B, 4):
        K, V = W.kv_tokens(4, s.Hkv, s.ctx, seed=s.seed + b0, device="cuda")
        kv.prefill(p, cache.slice(b0, b0 + 4), K, V)
        if b0 == 36:
            keep = {"K": K[1, 5].clone(), "V": V[1, 5].clone()}       # unit (37, 5)
        del K, V
    assert cache.seq_lens.tolist() == [s.ctx] * s.B
    q = W.queries(s.B, s.Hq, seed=s.seed, device="cuda")
    out = kv.decode_attention(p, cache, q)
    assert torch.isfinite(out).all()
    units = [(0, 0), (5, 2), (17, 6), (26, 1), (37, 5), (44, 3), (58, 4), (63, 7)]
    errs = _check_units(kv, p, cache, q, out, s.ctx, units)
    own = fanout.pmap("cache_attention", [(P.tile_f64(q[37, 5 * s.g:6 * s.g]), P.tile_f64(keep["K"]), P.tile_f64(keep["V"]), 0, bits)], 1)
    o = out[37, 5 * s.g:6 * s.g].double().cpu().numpy()
    drift, e_gpu, e_orc = P.attn_rel_err(o, own[0][0]), P.attn_rel_err(o, own[0][1]), P.attn_rel_err(own[0][0], own[0][1])
    print(f"configs[4] {bits}-bit: attention vs oracle max {max(errs):.2e} over {len(units)} units; end to end on unit (37, 5): "
          f"drift vs the oracle's own cache {drift:.1e}, error vs un-quantised attention GPU cache {e_gpu:.1e} / oracle cache {e_orc:.1e}")
    assert e_gpu <= 2.0 * e_orc + 1e-3 and drift <= 0.5


# ------------------------------------------------------------------------------------------------ adversarial
@pytest.mark.parametrize("bits", [2, 4])
def test_dominant_token_over_a_flat_64k_tail(kv, bits):
    """VERDICT r1 weak 3 / ADVICE 1: one token whose logit lies 24 (12, 30) log2 units above a flat tail of 65 535
    tokens.  Relative to the dominant token every tail probability is 2^-24 -- below the 2^-23 resolution of the
    22-bit fixed-point probabilities -- yet the tail holds 0.4 % of the mass and ALL of the output (the value rows
    of the dominant token's neighbourhood are zero).  The kernel's probabilities refer to the maximum of their own
    loop iteration (<= 256 tokens), so the tail is represented exactly whatever the context length; only tokens that
    share an iteration with the dominant one fall below the resolution (the bound kvarn.h states), hence the three
    chunks around it carry zero values here.  Records are hand-made through kvarn_pack_record_host:
    K_hat[t, :] = s2[t] * 1, so with q = a * e_0 the logit of token t is a * s2[t] nats."""
    p = kv.default_params(bits)
    lv = (1 << bits) - 1
    n_chunks, tstar = 512, 300 * 128 + 77
    ones, zeros = np.ones(128, dtype=np.float32), np.zeros(128, dtype=np.float32)
    k_plain = kv.pack_record(p, 0, np.ones((128, 128), dtype=np.uint8), ones, ones, zeros)
    s2 = ones.copy(); s2[tstar % 128] = 2.0
    k_star = kv.pack_record(p, 0, np.ones((128, 128), dtype=np.uint8), ones, s2, zeros)
    rng = np.random.default_rng(5)
    cache = kv.Cache(p, 1, 1, n_chunks, device="cuda")
    krec = np.tile(k_plain, (n_chunks, 1)); krec[tstar // 128] = k_star
    vrec = np.empty_like(krec)
    for c in range(n_chunks):
        codes = rng.integers(0, lv + 1, size=(128, 128)).astype(np.uint8)
        if abs(c - tstar // 128) <= 1:
            codes[:] = 0                                 # the dominant token's neighbourhood: zero value rows
        vrec[c] = kv.pack_record(p, 1, codes, ones, ones, zeros)
    cache.k_records[0, 0] = torch.tensor(krec, device="cuda")
    cache.v_records[0, 0] = torch.tensor(vrec, device="cuda")
    cache.seq_lens.fill_(n_chunks * 128)
    q = torch.zeros((1, 4, 128), device="cuda", dtype=torch.bfloat16)
    for h, a in enumerate((16.625, 8.3125, 20.75, 0.0)):     # 24, 12, 30 log2 units; flat
        q[0, h, 0] = a
    for splits in (0, 1, 8, 16):
        p.splits = splits
        out = kv.decode_attention(p, cache, q)
        errs = _check_units(kv, p, cache, q, out, n_chunks * 128, [(0, 0)])
        assert float(out[0, 0].abs().max()) > 0          # the tail's contribution is there


@pytest.mark.parametrize("offset,tol", [(50.0, 1.0), (500.0, 10.0)])
def test_channel_offsets_far_above_std(kv, offset, tol):
    """VERDICT r1 weak 3 / ADVICE 4: tiles whose channels carry offsets of 50 and 500 standard deviations (P:127
    "in some cases have large offsets"): the row variances of Alg. 1 must stay mean-centred in fp32 (the kernel
    switches such tiles to pivoted row passes).  At 50 the north_star tolerances hold as they are.  At 500 the fp32
    INPUT limits what any fp32 pipeline can do: values of size 500 sigma carry 2^-24 relative rounding through the
    seven butterfly stages of the rotation, i.e. ~1e-4 sigma of noise on every rotated element -- the data the
    quantizer sees differs from the oracle's float64 rotation by that much -- so scales are compared at 10 x 1e-5 and
    the code budget at 10 x 1e-4 (kvarn.h states the bound: tolerances hold up to |offset| / std ~ 100)."""
    p = kv.default_params(2)
    X = torch.stack([W.offset_tile(seed=11 + i, offset=offset, device="cuda") for i in range(4)])
    k_rec, v_rec, dbg = kv.quantize_chunk(p, X, X.clone(), debug=True)
    torch.cuda.synchronize()
    stats = {}
    for kind, R in enumerate((k_rec, v_rec)):
        P.check_quantized_tiles(kv, p, kind, list(X.double().cpu().numpy()), list(R.cpu().numpy()),
                                dbg.k_best[kind].cpu().numpy(), dbg.imb[kind].cpu().numpy(), dbg.aux[kind].cpu().numpy(), stats,
                                procs=1, tol=tol)
    P.assert_mismatch_budget(stats, aux_frac=P.AUX_MISMATCH_FRAC * tol * 30, code_frac=P.CODE_MISMATCH_FRAC * tol)
    print(f"offset {offset}: {stats}")


# ------------------------------------------------------------------------------------------------ aux ties
def test_storage_rounding_tie_rate_over_2000_tiles(kv):
    """stored FP8 / FP16 values may differ from the oracle's only where the pre-storage value sits
    on a rounding boundary.  Measured here over 2 x 1024 config-1-style tiles + 2 x 1024 config-3-style tiles
    (786 432 stored values per bit width): the rate must stay below the 1e-4 budget north_star gives the codes
    (DESIGN.md "Tolerances" derives the expected ~1e-5: the kernel's fp32 values agree with the oracle's to
    ~1e-7 relative, an FP16 zero-point has 2^10 boundaries per octave, an FP8 scale 2^3)."""
    K1, V1 = W.kv_tokens(1, 8, 128 * 128, seed=1, device="cuda")
    K3, V3 = W.quantizer_sweep_tiles(8, 128 * 128, seed=3, device="cuda")
    Kt = torch.cat([K1.reshape(-1, 128, 128), K3.reshape(-1, 128, 128)])
    Vt = torch.cat([V1.reshape(-1, 128, 128), V3.reshape(-1, 128, 128)])
    assert Kt.shape[0] == 2048
    for bits in (2, 4):
        p = kv.default_params(bits)
        stats = {}
        _check_tiles(kv, p, Kt, Vt, list(range(2048)), stats)
        rate = stats["aux_mismatch"] / stats["aux"]
        print(f"{bits}-bit: {stats}; aux tie rate {rate:.2e}, code tie rate {stats['code_mismatch'] / stats['codes']:.2e}")
        assert stats["tiles"] == 4096 and rate <= P.AUX_MISMATCH_FRAC
        P.assert_mismatch_budget(stats)


def _fill(kv, p, B, Hkv, ctx, seed):
    cache = kv.Cache(p, B, Hkv, ctx // 128 + 1, device="cuda")
    for b0 in range(0, B, 4):
        K, V = W.kv_tokens(min(4, B - b0), Hkv, ctx, seed=seed + b0, device="cuda")
        kv.prefill(p, cache.slice(b0, min(b0 + 4, B)), K, V)
        del K, V
    return cache


@pytest.mark.parametrize("n_q", [32, 128])
def test_block_attention_at_64k_context_in_the_bench_configuration(kv, n_q):
    """Both block-attention forms in the launch configuration bench.py times (B = 16, 32 / 8 heads, 65 536 + 37 tokens,
    2-bit; n_q = 32: one row tile per CTA, direct output; n_q = 128: four row tiles x two chunk ranges + merge for the
    dense kernel): sampled (sequence, KV head, query token) triples against the oracle's plain-definition attention of
    that query over the GPU's records, the raw residual tokens and the block tokens it may see (causal); the dense and
    the integer form against each other on every row."""
    B, Hq, Hkv, ctx = 16, 32, 8, 65536 + 37
    g = Hq // Hkv
    p = kv.default_params(2)
    cache = _fill(kv, p, B, Hkv, ctx, seed=77)
    q = torch.stack([W.queries(B, Hq, seed=900 + i, device="cuda") for i in range(n_q)], dim=1).contiguous()
    kb, vb = W.kv_tokens(B, Hkv, n_q, seed=950, device="cuda", sink_first=False)
    dense = kv.block_attention(p, cache, q, kb, vb, dense=True)
    triples = [(0, 0, 0), (7, 3, n_q // 2), (15, 7, n_q - 1)]
    jobs = []
    for b, h, i in triples:
        ns, nc, r = O.cache_partition(ctx, cache.n_sink)
        kt = [kv.unpack_record(p, 0, rec) for rec in cache.k_records[b, h, :nc].cpu().numpy()]
        vt = [kv.unpack_record(p, 1, rec) for rec in cache.v_records[b, h, :nc].cpu().numpy()]
        kraw = np.concatenate([P.tile_f64(cache.k_resid[b, h, :r]), P.tile_f64(kb[b, h, :i + 1])])
        vraw = np.concatenate([P.tile_f64(cache.v_resid[b, h, :r]), P.tile_f64(vb[b, h, :i + 1])])
        jobs.append((P.tile_f64(q[b, i, h * g:(h + 1) * g]), kt, vt, kraw, vraw, None, True, True))
    refs = fanout.pmap("decode", jobs)
    forms = {"dense": dense}
    if n_q == 32:                                   # the integer form costs 140 us per query token: only on the smaller block
        forms["integer"] = kv.block_attention(p, cache, q, kb, vb)
    for name, out in forms.items():
        o = out.to(torch.float64).cpu().numpy()
        for (b, h, i), ref in zip(triples, refs):
            err = P.attn_rel_err(o[b, i, h * g:(h + 1) * g], ref)
            assert err <= P.ATTN_RTOL, (name, b, h, i, err)
    if n_q == 32:
        d = (forms["dense"].double() - forms["integer"].double()).abs().amax(dim=-1)
        scale = forms["integer"].double().abs().amax(dim=-1).clamp_min(1e-30)
        assert float((d / scale).max()) <= P.ATTN_RTOL
