"""GPU parity: kvarn_quantize_chunk (through the C ABI) vs the oracle, element by
element on the same seeded inputs (BASELINE.json configs 0 and 3, edge cases)."""
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


def _run_and_check(kv, p, K, V, stats=None):
    """K, V torch [n, 128, 128] on cuda.  Checks every tile of both kinds."""
    k_rec, v_rec, dbg = kv.quantize_chunk(p, K, V, debug=True)
    torch.cuda.synchronize()
    stats = {} if stats is None else stats
    kb, imb, aux = dbg.k_best.cpu().numpy(), dbg.imb.cpu().numpy(), dbg.aux.cpu().numpy()
    recs = (k_rec.cpu().numpy(), v_rec.cpu().numpy())
    for kind, X in ((0, K), (1, V)):
        for i in range(X.shape[0]):
            P.check_quantized_tile(kv, p, kind, P.tile_f64(X[i]), recs[kind][i], int(kb[kind, i]),
                                   imb[kind, i], aux[kind, i], stats)
    return stats, recs, kb


def test_config0_single_tile_fp32(kv):
    # BASELINE.json configs[0]: K with 4 outlier channels x20 and token 0 x10
    K, V, q, oc = W.config0()
    p = kv.default_params(2)
    Kt, Vt = torch.tensor(K, device="cuda")[None], torch.tensor(V, device="cuda")[None]
    stats, recs, kb = _run_and_check(kv, p, Kt, Vt)
    P.assert_mismatch_budget(stats)
    assert recs[0].shape == (1, 4608)
    # token 0 (x10) carries the largest per-token second scale of the K tile
    _, _, s2, _ = kv.unpack_record(p, 0, recs[0][0])
    assert int(np.argmax(s2)) == 0


@pytest.mark.parametrize("bits", [2, 4])
def test_config3_sample_bf16(kv, bits):
    # config 3 recipe (log-normal channel scales, 1 % token outliers x8), a
    # multi-tile launch spanning several waves' worth of CTAs with a ragged count
    K, V = W.quantizer_sweep_tiles(Hkv=8, n_tok=128 * 37, seed=3, device="cuda")
    Kt = K.reshape(-1, 128, 128).contiguous()
    Vt = V.reshape(-1, 128, 128).contiguous()
    assert Kt.shape[0] == 296
    p = kv.default_params(bits)
    k_rec, v_rec, dbg = kv.quantize_chunk(p, Kt, Vt, debug=True)
    torch.cuda.synchronize()
    kb, imb, aux = dbg.k_best.cpu().numpy(), dbg.imb.cpu().numpy(), dbg.aux.cpu().numpy()
    recs = (k_rec.cpu().numpy(), v_rec.cpu().numpy())
    stats = {}
    rng = np.random.default_rng(0)
    sample = sorted(set([0, 1, 147, 148, 295]) | set(rng.choice(296, 19, replace=False).tolist()))
    for kind, X in ((0, Kt), (1, Vt)):
        for i in sample:
            P.check_quantized_tile(kv, p, kind, P.tile_f64(X[i]), recs[kind][i], int(kb[kind, i]),
                                   imb[kind, i], aux[kind, i], stats)
    P.assert_mismatch_budget(stats)


# configs[3] at full size (131 072 tiles per kind, >= 1 % of them against the oracle): tests/test_gpu_parity_full.py


def test_deterministic_and_k_only_v_only(kv):
    K, V = W.quantizer_sweep_tiles(Hkv=2, n_tok=128 * 3, seed=5, device="cuda")
    Kt, Vt = K.reshape(-1, 128, 128).contiguous(), V.reshape(-1, 128, 128).contiguous()
    p = kv.default_params(2)
    a = kv.quantize_chunk(p, Kt, Vt)
    b = kv.quantize_chunk(p, Kt, Vt)
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
    ko, _ = kv.quantize_chunk(p, Kt, None)
    _, vo = kv.quantize_chunk(p, None, Vt)
    assert torch.equal(ko, a[0]) and torch.equal(vo, a[1])


def test_offset_tile_variance_is_mean_centred(kv):
    # P:127 "in some cases have large offsets": channels with mean >> std
    X = W.offset_tile(seed=11, offset=6.0, device="cuda")
    p = kv.default_params(2)
    stats, _, _ = _run_and_check(kv, p, X[None], X[None].clone())
    P.assert_mismatch_budget(stats)


@pytest.mark.parametrize("opts", [dict(iters=0), dict(iters=1), dict(iters=3), dict(rotate_k=0, rotate_v=0),
                                  dict(iters=0, rotate_k=0, rotate_v=0)])
def test_ablation_switches(kv, opts):
    # KIVI (RTN only), HK (Hadamard + RTN), VarN(K) -- the same kernel with flags
    K, V, _, _ = W.config0()
    p = kv.default_params(2, **opts)
    Kt, Vt = torch.tensor(K, device="cuda")[None], torch.tensor(V, device="cuda")[None]
    stats, _, kb = _run_and_check(kv, p, Kt, Vt)
    P.assert_mismatch_budget(stats)
    if p.iters == 0:
        assert kb.max() == 0


def test_degenerate_tiles_do_not_fault(kv):
    p = kv.default_params(2)
    Z = torch.zeros((1, 128, 128), device="cuda", dtype=torch.bfloat16)
    Cst = torch.full((1, 128, 128), 1.5, device="cuda", dtype=torch.bfloat16)
    for X in (Z, Cst):
        k_rec, v_rec = kv.quantize_chunk(p, X, X.clone())
        torch.cuda.synchronize()
        for kind, rec in ((0, k_rec), (1, v_rec)):
            codes, s1, s2, z = kv.unpack_record(p, kind, rec[0].cpu().numpy())
            assert np.isfinite(s1).all() and np.isfinite(s2).all() and np.isfinite(z).all()
    # all-zero tile: every variance 0 -> clamped, L = -0.3 on both axes; RTN
    # groups degenerate -> codes 0, z = 0, dequant = 0 exactly
    codes, s1, s2, z = kv.unpack_record(p, 0, kv.quantize_chunk(p, Z, Z.clone())[0][0].cpu().numpy())
    assert codes.sum() == 0 and np.all(z == 0)
    # non-finite input: undefined values, no fault
    X = torch.randn((2, 128, 128), device="cuda").to(torch.bfloat16)
    X[0, 3, 7] = float("inf"); X[1, 5, 5] = float("nan")
    kv.quantize_chunk(p, X, X.clone())
    torch.cuda.synchronize()


def test_strided_input_and_record_stride(kv):
    # tokens of a tile need not be contiguous with the next tile: [Hkv][n_tok][128]
    # viewed per head with a padded token stride
    import ctypes as C
    K, V = W.quantizer_sweep_tiles(Hkv=1, n_tok=128 * 4, seed=9, device="cuda")
    pad = torch.zeros((4 * 128, 256), device="cuda", dtype=torch.bfloat16)
    pad[:, :128] = K[0]
    p = kv.default_params(2)
    rec_s = torch.zeros((4, 4608 + 64), dtype=torch.uint8, device="cuda")
    st = kv.lib.kvarn_quantize_chunk(C.byref(p), C.c_void_p(pad.data_ptr()), None, 4, 128 * 256, 256,
                                     C.c_void_p(rec_s.data_ptr()), None, 4608 + 64, None,
                                     C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert st == 0
    ref, _ = kv.quantize_chunk(p, K[0].reshape(4, 128, 128).contiguous(), None)
    torch.cuda.synchronize()
    assert torch.equal(rec_s[:, :4608], ref) and int(rec_s[:, 4608:].sum()) == 0


def test_zero_tiles_is_a_noop(kv):
    p = kv.default_params(2)
    E = torch.empty((0, 128, 128), device="cuda", dtype=torch.bfloat16)
    k_rec, v_rec = kv.quantize_chunk(p, E, E.clone())
    assert k_rec.shape == (0, 4608)


def test_quantize_is_deterministic_over_repeats(kv):
    # same reasoning as the decode repeat test: identical launches must give identical bytes
    K, V = W.quantizer_sweep_tiles(8, 128 * 64, seed=5, device="cuda")
    Kt, Vt = K.reshape(-1, 128, 128), V.reshape(-1, 128, 128)
    for bits in (2, 4):
        p = kv.default_params(bits)
        k0, v0 = kv.quantize_chunk(p, Kt, Vt)
        for _ in range(20):
            k1, v1 = kv.quantize_chunk(p, Kt, Vt)
            assert torch.equal(k0, k1) and torch.equal(v0, v1)


def test_error_decomposition_ranks_the_ablations(kv):
    # SURVEY 8(f3) / P:25 Fig. 1b, Eq. 2-3: on K tiles with channel outliers AND high-norm tokens the
    # per-token magnitude error E_M of KVarN (Hadamard + VarN + RTN) is far below both HK's (Hadamard + RTN) and
    # KIVI's (RTN only) -- on this data the oracle gives E_M = 86 / 2619 / 1832.  Records come from the CUDA
    # quantizer in its three flag settings; dequantisation (Eq. 1) and the decomposition E_T = E_M + E_D are the
    # oracle's.  A soft, qualitative check on synthetic data: it gates only "KVarN at most half of the others"
    # (the order of HK and KIVI among themselves depends on the data and is not asserted).
    g = torch.Generator(device="cpu"); g.manual_seed(17)
    n = 32
    K = torch.randn((n, 128, 128), generator=g)
    K[:, :, torch.randperm(128, generator=g)[:4]] *= 20.0            # channel outliers
    tok = torch.rand((n, 128, 1), generator=g) < 0.05
    K = (K * torch.where(tok, torch.tensor(8.0), torch.tensor(1.0))).to(torch.bfloat16).cuda()
    Kf = K.double().cpu().numpy()
    res = {}
    for name, opts in (("kivi", dict(iters=0, rotate_k=0, rotate_v=0)), ("hk", dict(iters=0)), ("kvarn", dict())):
        p = kv.default_params(2, **opts)
        rec, _ = kv.quantize_chunk(p, K, None)
        em = et = 0.0
        for i in range(n):
            codes, s1, s2, z = kv.unpack_record(p, 0, rec[i].cpu().numpy())
            Kdq = O.dequantize_tile(codes, s1.astype(np.float64), s2.astype(np.float64), z.astype(np.float64), "k",
                                    rotate_on=bool(p.rotate_k))
            E_T, E_M, E_D = O.error_decomposition(Kf[i], Kdq)
            assert np.allclose(E_T, E_M + E_D, rtol=1e-9, atol=1e-9)      # Eq. 3
            em += float(E_M.mean()); et += float(E_T.mean())
        res[name] = (em / n, et / n)
    for other in ("hk", "kivi"):
        assert res["kvarn"][0] < 0.5 * res[other][0], res     # magnitude error E_M
        assert res["kvarn"][1] < 0.5 * res[other][1], res     # total error E_T


@pytest.mark.parametrize("bits", [2, 4])
def test_round_before_variant_vs_oracle(kv, bits):
    """aux_round = 1 (reading R9b): RTN against the stored FP8 / FP16 parameters."""
    n = 48
    K, V = W.quantizer_sweep_tiles(8, n * 128 // 8, seed=17, device="cuda")
    Kt, Vt = K.reshape(n, 128, 128), V.reshape(n, 128, 128)
    p = kv.default_params(bits, aux_round=1)
    kr, vr, dbg = kv.quantize_chunk(p, Kt, Vt, debug=True)
    stats = {}
    for kind, (T, R) in enumerate(((Kt, kr), (Vt, vr))):
        for i in range(0, n, 3):
            P.check_quantized_tile(kv, p, kind, P.tile_f64(T[i]), R[i].cpu().numpy(), int(dbg.k_best[kind, i]),
                                   dbg.imb[kind, i].cpu().numpy(), dbg.aux[kind, i].cpu().numpy(), stats)
    # R9b: z = fp16(mn / (fp8(s1) / absorbed)) -- a quotient of rounded quantities -- lands on an FP16 boundary more
    # often than the plain z = mn / s: measured 3 of 6144 zero-points here, against 9e-5 per zero-point in the default mode
    P.assert_mismatch_budget(stats, aux_frac=3e-4)
    # the variant's purpose: dequantising the stored record reproduces the token norms better at 4-bit
    if bits == 4:
        p0 = kv.default_params(bits)
        kr0, _ = kv.quantize_chunk(p0, Kt, Vt)
        def tokmag(rec, i):
            X = P.tile_f64(Kt[i])
            Xd = O.dequantize_tile(*[np.asarray(a, dtype=np.float64) for a in kv.unpack_record(p, 0, rec[i].cpu().numpy())], kind="k")
            return np.mean(np.abs(np.linalg.norm(Xd, axis=1) / np.linalg.norm(X, axis=1) - 1))
        a = np.mean([tokmag(kr, i) for i in range(6)]); b = np.mean([tokmag(kr0, i) for i in range(6)])
        assert a < 0.6 * b, (a, b)


def test_round_before_decode_matches_oracle_on_its_records(kv):
    """The read path is unchanged by aux_round: a cache written with either setting decodes to the oracle's
    attention over those records."""
    K, V = W.kv_tokens(1, 2, 128 * 4, seed=19, device="cuda")
    q = W.queries(1, 8, seed=19, device="cuda")
    for ar in (0, 1):
        p = kv.default_params(4, aux_round=ar)
        cache = kv.Cache(p, 1, 2, 4)
        kv.prefill(p, cache, K, V)
        out = kv.decode_attention(p, cache, q).double().cpu().numpy()
        worst = 0.0
        for h in range(2):
            ref = P.oracle_attention_from_records(kv, p, cache.k_records[0, h].cpu().numpy(), cache.v_records[0, h].cpu().numpy(),
                                                  np.zeros((0, 128)), np.zeros((0, 128)), P.tile_f64(q[0, 4 * h:4 * h + 4]))
            worst = max(worst, P.attn_rel_err(out[0, 4 * h:4 * h + 4], ref))
        assert worst <= P.ATTN_RTOL, worst


@pytest.mark.parametrize("bits", [2, 4])
def test_adversarial_tiles_vs_oracle(kv, bits):
    """Tiles built to stress the normaliser and the storage formats, against the oracle at the iterate the kernel kept:
    token norms over 16 binades, channel norms over 12 binades (the log clamps of Alg. 1 bind), one element 2^14 above
    the rest, exact-zero rows and columns, and a tile of magnitude 2^-40."""
    g = torch.Generator(device="cuda").manual_seed(31 + bits)
    base = torch.randn((5, 128, 128), generator=g, device="cuda")
    T = base.clone()
    T[0] *= torch.exp2(torch.randint(-8, 9, (128, 1), generator=g, device="cuda").float())      # token norms
    T[1] *= torch.exp2(torch.randint(-6, 7, (1, 128), generator=g, device="cuda").float())      # channel norms
    T[2, 17, 93] = 2.0 ** 14                                                                       # one massive element
    T[3, 5::19, :] = 0; T[3, :, 7::23] = 0                                                         # zero rows and columns
    T[4] *= 2.0 ** -40            # small magnitudes (fp32 variances: below ~2^-60 the squares underflow, kvarn.h states the bound)
    X = T.to(torch.bfloat16)
    p = kv.default_params(bits)
    stats, recs, kb = _run_and_check(kv, p, X, X.flip(0).contiguous())
    P.assert_mismatch_budget(stats, aux_frac=3e-4)
    for kind in (0, 1):
        for rec in recs[kind]:
            codes, s1, s2, z = kv.unpack_record(p, kind, rec)
            assert np.isfinite(s1).all() and np.isfinite(s2).all() and np.isfinite(z).all()
