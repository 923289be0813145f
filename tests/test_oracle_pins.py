"""Pins for oracle/kvarn_oracle.py against what the paper and mathematics fix.

None of these re-types the oracle's own formula: each compares against a closed
form, a library routine, an invariant, brute force, or a textbook special case,
chosen so that a dropped term, a wrong sign / axis / index or a transposed
operand in the oracle fails at least one.  Citations ``P:n`` = PAPER.md line n.
"""
import math

import numpy as np
import pytest
import scipy.linalg
import torch

from oracle import kvarn_oracle as O
from paper_2606_03458_b200 import workloads as W


# ----------------------------------------------------------------- Hadamard
def test_hadamard_is_scipy_sylvester():
    # library routine: scipy's Sylvester construction
    for d in (2, 8, 128):
        assert np.array_equal(O.hadamard_matrix(d), scipy.linalg.hadamard(d).astype(np.float64))


def test_hadamard_orthogonal_symmetric():
    H = O.hadamard_matrix(128)
    assert np.array_equal(H @ H.T, 128 * np.eye(128))      # H H^T = d I
    assert np.array_equal(H, H.T)
    assert set(np.unique(H)) == {-1.0, 1.0}


def test_rotate_is_rotation_along_channels():
    rng = np.random.default_rng(5)
    X = rng.standard_normal((7, 128))
    Y = O.rotate(X)
    # norm of every TOKEN preserved (rotation along the channel axis)
    assert np.allclose(np.linalg.norm(Y, axis=1), np.linalg.norm(X, axis=1), rtol=1e-13)
    # involution: H/sqrt(d) is its own inverse
    assert np.allclose(O.rotate(Y), X, atol=1e-13)
    # channel axis, not token axis: a one-hot token maps to a +-1/sqrt(d) row
    e = np.zeros((3, 128)); e[1, 5] = 1.0
    Ye = O.rotate(e)
    assert np.allclose(np.abs(Ye[1]), 1 / math.sqrt(128)) and np.all(Ye[0] == 0) and np.all(Ye[2] == 0)
    # channel 0 of the output is the scaled sum (first Sylvester row is all ones)
    assert np.allclose(Y[:, 0], X.sum(axis=1) / math.sqrt(128))
    # inner products preserved => q'.k' = q.k (what decode attention relies on)
    q = rng.standard_normal((2, 128))
    assert np.allclose(O.rotate(q) @ Y.T, q @ X.T, atol=1e-12)


# --------------------------------------------------------------------- VarN
def _balanced_E(seed=0):
    """E = [[A, -A], [-A, A]], A in {+-1}^(64x64): every row and column has
    mean 0 and population variance exactly 1."""
    rng = np.random.default_rng(seed)
    A = rng.choice([-1.0, 1.0], size=(64, 64))
    return np.block([[A, -A], [-A, A]])


def test_varn_closed_form_column_scales():
    # T = E diag(b): after ONE iteration S_c = b, S_r = 1, I = 1 exactly.
    # Pins: update axis order (columns = tokens first), the 1/2 factor,
    # population variance (ddof=1 would give b*sqrt(128/127)), division (not
    # multiplication) by the scales, and the "<=" keep rule.
    E = _balanced_E(1)
    rng = np.random.default_rng(2)
    b = np.exp(rng.uniform(-0.25, 4.0, size=128))
    r = O.varn(E * b[None, :], iters=1)
    assert np.allclose(r.S_c, b, rtol=1e-12)
    assert np.allclose(r.S_r, 1.0, rtol=1e-12)
    assert abs(r.I[1] - 1.0) < 1e-12 and r.k_best == 1
    assert np.allclose(r.T_bal, E, atol=1e-12)
    # stays there for more iterations
    r8 = O.varn(E * b[None, :], iters=8)
    assert np.allclose(r8.S_c, b, rtol=1e-12) and np.allclose(r8.S_r, 1.0, rtol=1e-12)


def test_varn_row_scales_need_second_half_step():
    # T = diag(a) E with a > e^-0.3: the column step sees v_col = mean(a^2)
    # (E^2 = 1), the row step then fixes each row exactly:
    # S_c = sqrt(mean a^2) (all equal), S_r = a / sqrt(mean a^2).
    E = _balanced_E(3)
    rng = np.random.default_rng(4)
    a = np.exp(rng.uniform(0.0, 0.5, size=128))
    r = O.varn(a[:, None] * E, iters=1)
    # column means of diag(a)E are not zero in general, so compute the exact
    # column variance by brute force instead of assuming mean(a^2)
    T = a[:, None] * E
    vcol = np.array([np.mean((T[:, t] - T[:, t].mean()) ** 2) for t in range(128)])
    S_c = np.sqrt(vcol)
    C1 = T / S_c[None, :]
    vrow = np.array([np.mean((C1[c] - C1[c].mean()) ** 2) for c in range(128)])
    assert np.allclose(r.S_c_k[1], S_c, rtol=1e-12)
    assert np.allclose(r.S_r_k[1], np.sqrt(vrow), rtol=1e-12)
    # after an unclamped row step every row variance is exactly 1
    C = T / r.S_c_k[1][None, :] / r.S_r_k[1][:, None]
    assert np.allclose(C.var(axis=1), 1.0, rtol=1e-12)


def test_varn_log_clamps():
    # P:445 / P:451: L clamped to [-0.3, 10].  T = 0.05 E => S = e^-0.3 both axes
    E = _balanced_E(5)
    r = O.varn(0.05 * E, iters=3)
    for k in (1, 2, 3):
        assert np.allclose(r.S_c_k[k], math.exp(-0.3)) and np.allclose(r.S_r_k[k], math.exp(-0.3))
    # T = 1e6 E: variance 1e12 hits c_max = 1e8 first => S_c = sqrt(1e8) = 1e4
    r = O.varn(1e6 * E, iters=1)
    assert np.allclose(r.S_c_k[1], 1e4)
    # with c_max out of the way the log clamp binds: ln(1e6) = 13.8 > 10
    r = O.varn(1e6 * E, iters=1, c_max=1e30)
    assert np.allclose(r.S_c_k[1], math.exp(10.0))
    # trajectory always inside the clamps
    K, V, _, _ = W.config0()
    rk = O.varn(O.rotate(K).T)
    for k in range(9):
        assert np.all(np.log(rk.S_c_k[k]) >= -0.3 - 1e-12) and np.all(np.log(rk.S_c_k[k]) <= 10 + 1e-12)
        assert np.all(np.log(rk.S_r_k[k]) >= -0.3 - 1e-12)


def test_varn_variance_clamp_constant_row():
    # c_min keeps log finite: a constant row has variance 0 -> clamp 1e-8 ->
    # 0.5 ln 1e-8 = -9.2 -> L = -0.3; output finite.
    E = _balanced_E(6)
    T = E.copy(); T[7, :] = 2.5
    r = O.varn(T, iters=2)
    assert np.isfinite(r.T_bal).all()
    assert np.isclose(r.S_r_k[1][7], math.exp(-0.3))


def test_varn_k0_identity_and_best_monotone():
    K, V, _, _ = W.config0()
    T = O.rotate(K).T
    r0 = O.varn(T, iters=0)
    assert np.all(r0.S_c == 1) and np.all(r0.S_r == 1) and np.array_equal(r0.T_bal, T)
    r = O.varn(T)
    # the kept imbalance is the minimum of the trajectory, "<=" keeps the LAST minimiser
    I = np.array(r.I)
    assert r.k_best == max(np.flatnonzero(I == I.min()))
    assert np.allclose(r.T_bal, T / r.S_c_k[r.k_best][None, :] / r.S_r_k[r.k_best][:, None])
    # T_bal * S_c * S_r reconstructs T (line 24 of Alg. 1 divides by both)
    assert np.allclose(r.T_bal * r.S_c[None, :] * r.S_r[:, None], T, rtol=1e-13)


def test_varn_uniform_variances_config0():
    # "Before quantization, the variance of the token and channel
    # dimensions of these normalized matrices are uniform."
    K, V, _, _ = W.config0()
    for X in (K, V):
        r = O.varn(O.rotate(X).T)
        vr, vc = r.T_bal.var(axis=1), r.T_bal.var(axis=0)
        allv = np.concatenate([vr, vc])
        assert allv.max() / allv.min() < 1.01
    # and the raw K tile is far from it (token 0 x10, P:25 token-scale outliers)
    T = O.rotate(K).T
    assert O.imbalance(T) > 100


def test_varn_axis_orientation_matters_and_is_token_first():
    # Reading R5: rows = channels, columns = tokens, column (token) scales
    # updated first.  On config-0 K the literal orientation converges, the
    # transposed one is stuck behind the -0.3 floor.
    K, _, _, _ = W.config0()
    Y = O.rotate(K)
    r_lit = O.varn(Y.T)
    r_swp = O.varn(Y)
    assert r_lit.I[8] < 1.01 < 2.0 < r_swp.I[8]
    # S_c is per token: the x10 token 0 gets by far the largest column scale
    assert np.argmax(r_lit.S_c) == 0 and r_lit.S_c[0] > 5 * np.median(r_lit.S_c)


def test_imbalance_formula_small():
    # reading R1 on a hand-computed 2x2: rows [1,3],[2,2]
    C = np.array([[1.0, 3.0], [2.0, 2.0]])
    # row variances: 1, 0 ; column variances: 0.25, 0.25 ; min 0 -> c_min
    assert O.imbalance(C, c_min=0.5) == pytest.approx(1.0 / 0.5)
    assert O.imbalance(_balanced_E(0)) == pytest.approx(1.0)
    # scale invariance of a ratio of variances
    rng = np.random.default_rng(0)
    X = rng.standard_normal((16, 16))
    assert O.imbalance(3.7 * X) == pytest.approx(O.imbalance(X))
    assert O.imbalance(X.T) == pytest.approx(O.imbalance(X))


# ---------------------------------------------------------------------- RTN
@pytest.mark.parametrize("bits", [2, 4])
@pytest.mark.parametrize("axis", [0, 1])
def test_rtn_on_grid_round_trip_exact(bits, axis):
    # X = (Q + z) * s with dyadic s, z and every group holding 0 and Lv
    # => codes == Q and Eq. 1 reproduces X exactly.
    Lv = (1 << bits) - 1
    rng = np.random.default_rng(bits * 10 + axis)
    Q = rng.integers(0, Lv + 1, size=(128, 128))
    if axis == 1:
        Q[:, 0], Q[:, 1] = 0, Lv
    else:
        Q[0, :], Q[1, :] = 0, Lv
    s = 2.0 ** rng.integers(-3, 4, size=128)
    z = rng.integers(-8, 9, size=128) / 4.0
    sh = (128, 1) if axis == 1 else (1, 128)
    X = (Q + z.reshape(sh)) * s.reshape(sh)
    codes, s_o, z_o = O.rtn_quantize(X, bits, group_axis=axis)
    assert np.array_equal(codes, Q)
    assert np.array_equal(s_o, s) and np.array_equal(z_o, z)
    assert np.array_equal(O.rtn_dequantize(codes, s_o, z_o, axis), X)


def test_rtn_is_textbook_minmax_quantizer():
    # independent 5-line per-group min-max quantizer, python loop
    rng = np.random.default_rng(9)
    X = rng.standard_normal((6, 128)) * rng.uniform(0.5, 4, size=(6, 1)) + rng.uniform(-2, 2, size=(6, 1))
    codes, s, z = O.rtn_quantize(X, 2, group_axis=1)
    for r in range(6):
        lo, hi = X[r].min(), X[r].max()
        step = (hi - lo) / 3
        ref = np.clip(np.round((X[r] - lo) / step), 0, 3)     # ties are measure-zero here
        assert np.array_equal(codes[r], ref)
        assert s[r] == pytest.approx(step) and z[r] * s[r] == pytest.approx(lo)
        # Eq. 1: (K_q + z) * s ; error bounded by half a step
        deq = (codes[r] + z[r]) * s[r]
        assert np.abs(deq - X[r]).max() <= step / 2 + 1e-12
        assert deq.min() == pytest.approx(lo) and deq.max() == pytest.approx(hi)


def test_rtn_half_to_even_and_degenerate():
    # group [0, 0.5, 1.5, 2.5, 3] has s = 1, z = 0: ties go to even
    X = np.array([[0.0, 0.5, 1.5, 2.5, 3.0]])
    codes, s, z = O.rtn_quantize(X, 2, group_axis=1)
    assert codes.tolist() == [[0, 0, 2, 2, 3]] and s[0] == 1 and z[0] == 0
    # degenerate (constant) group: s = 1, codes 0, z = value (reading R7)
    codes, s, z = O.rtn_quantize(np.full((1, 8), -1.25), 2, group_axis=1)
    assert codes.sum() == 0 and s[0] == 1 and z[0] == -1.25
    assert np.array_equal(O.rtn_dequantize(codes, s, z, 1), np.full((1, 8), -1.25))


def test_k_per_channel_v_per_token_grouping():
    # "quantize the V matrix per token and the K matrix per channel".
    # With rotation and VarN off the tile quantizer is plain KIVI RTN.
    rng = np.random.default_rng(12)
    X = rng.standard_normal((128, 128))
    tk = O.quantize_tile(X, "k", iters=0, rotate_on=False)
    tv = O.quantize_tile(X, "v", iters=0, rotate_on=False)
    # K: channel c group spans the tokens -> every COLUMN of codes[t, c] hits 0 and 3
    assert np.all(tk.codes.min(axis=0) == 0) and np.all(tk.codes.max(axis=0) == 3)
    # V: token t group spans the channels -> every ROW hits 0 and 3
    assert np.all(tv.codes.min(axis=1) == 0) and np.all(tv.codes.max(axis=1) == 3)
    # scale of K channel 5 = (max - min over tokens) / 3
    assert tk.s1_f[5] == pytest.approx((X[:, 5].max() - X[:, 5].min()) / 3)
    assert tv.s1_f[5] == pytest.approx((X[5, :].max() - X[5, :].min()) / 3)
    assert np.all(tk.s2_f == 1) and np.all(tv.s2_f == 1)


# ---------------------------------------------------------------------- aux
def test_fp8_e4m3_matches_torch_cast():
    # library routine: torch's float8_e4m3fn cast (RNE).  Range kept < 448
    # where torch and the saturating definition agree.
    rng = np.random.default_rng(3)
    x = np.concatenate([
        np.exp(rng.uniform(np.log(2.0 ** -11), np.log(447.0), size=20000)),
        -np.exp(rng.uniform(np.log(2.0 ** -9), np.log(447.0), size=2000)),
        np.array([0.0, 2.0 ** -9, 2.0 ** -10, 3 * 2.0 ** -10, 448.0, 0.0175, 1.0625, 1.1875, 17.0, 19.0]),
    ])
    ref = torch.tensor(x, dtype=torch.float32).to(torch.float8_e4m3fn)
    got = O.round_fp8_e4m3(x.astype(np.float32).astype(np.float64))
    assert np.array_equal(got, ref.to(torch.float64).numpy())
    # byte encoding round trip, against torch's bytes
    bits = O.fp8_e4m3_bits(got)
    assert np.array_equal(bits, ref.view(torch.uint8).numpy())
    assert np.array_equal(O.fp8_e4m3_from_bits(bits), got)
    # every one of the 254 finite bytes decodes as torch decodes it
    allb = np.array([b for b in range(256) if (b & 0x7F) != 0x7F], dtype=np.uint8)
    tv = torch.tensor(allb).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert np.array_equal(O.fp8_e4m3_from_bits(allb), tv)


def test_fp8_saturates():
    assert O.round_fp8_e4m3(np.array([1e5, -1e5, 460.0, 448.0])).tolist() == [448.0, -448.0, 448.0, 448.0]


def test_fp16_matches_torch_cast():
    rng = np.random.default_rng(4)
    x = rng.standard_normal(5000) * np.exp(rng.uniform(-8, 8, size=5000))
    ref = torch.tensor(x, dtype=torch.float64).to(torch.float16).to(torch.float64).numpy()
    assert np.array_equal(O.round_fp16(x), ref)


def test_bit_accounting_2_25_bits_per_element():
    # 2 bits + two FP8 scales + one FP16 zero per 128 elements = 2.25
    K, V, _, _ = W.config0()
    nbytes = 0
    for X, kind in ((K, "k"), (V, "v")):
        t = O.quantize_tile(X, kind)
        nbytes += t.codes.size * 2 // 8 + t.s1.size * 1 + t.s2.size * 1 + t.z.size * 2
    assert nbytes == 9216
    assert nbytes * 8 / (2 * 128 * 128) == 2.25


def test_absorbed_and_second_scale_assignment():
    # P:382 "one of which absorbs the Sinkhorn normalisation scale into the RTN
    # scale"; reading R8: the absorbed one is constant along the RTN group.
    K, V, _, _ = W.config0()
    tk = O.quantize_tile(K, "k")
    tv = O.quantize_tile(V, "v")
    # second scale = the OTHER Sinkhorn scale, untouched by RTN
    assert np.array_equal(tk.s2_f, tk.varn.S_c)      # K: per token
    assert np.array_equal(tv.s2_f, tv.varn.S_r)      # V: per channel
    # absorbed: s1 / Sinkhorn scale is the plain RTN step of the balanced tile
    stepk = (tk.varn.T_bal.max(axis=1) - tk.varn.T_bal.min(axis=1)) / 3
    assert np.allclose(tk.s1_f / tk.varn.S_r, stepk, rtol=1e-12)
    stepv = (tv.varn.T_bal.max(axis=0) - tv.varn.T_bal.min(axis=0)) / 3
    assert np.allclose(tv.s1_f / tv.varn.S_c, stepv, rtol=1e-12)
    # token 0 of K (x10) carries its magnitude in the per-token second scale
    assert np.argmax(tk.s2) == 0


def test_dequant_eq1_with_second_scale_unrounded_is_rtn_error_only():
    # with UNROUNDED aux, dual-scale dequant = T_bal's RTN error mapped back:
    # |Yhat - Y|[t,c] <= (s/2) * S_c[t] * S_r[c]   (Eq. 1 + P:125)
    K, V, _, _ = W.config0()
    for X, kind in ((K, "k"), (V, "v")):
        t = O.quantize_tile(X, kind)
        Yhat = O.dequantize_tile(t.codes, t.s1_f, t.s2_f, t.z_f, kind, rotate_on=False)
        Y = O.rotate(X)
        if kind == "k":
            bound = 0.5 * t.s1_f[None, :] * t.s2_f[:, None]
        else:
            bound = 0.5 * t.s1_f[:, None] * t.s2_f[None, :]
        assert np.all(np.abs(Yhat - Y) <= bound * (1 + 1e-9) + 1e-12)
        # and the full route returns to the un-rotated space
        Xd = O.dequantize_tile(t.codes, t.s1_f, t.s2_f, t.z_f, kind)
        assert np.allclose(O.rotate(Xd), Yhat, atol=1e-12)


def test_kvarn_beats_plain_rtn_on_token_magnitude_soft():
    # Soft sanity check of the paper's qualitative claim (Fig. 1b), on the
    # synthetic outlier tile only: per-token magnitude error of KVarN < KIVI.
    K, _, _, _ = W.config0()
    def mag_err(**kw):
        t = O.quantize_tile(K, "k", **kw)
        Kd = O.dequantize_tile(t.codes, t.s1, t.s2, t.z, "k", rotate_on=kw.get("rotate_on", True))
        return np.abs(np.linalg.norm(Kd, axis=1) / np.linalg.norm(K, axis=1) - 1).mean()
    assert mag_err() < mag_err(iters=0, rotate_on=False)


def test_error_decomposition_identity():
    # Eq. 3: E_T = E_M + E_D
    rng = np.random.default_rng(1)
    A, B = rng.standard_normal((9, 128)), rng.standard_normal((9, 128))
    E_T, E_M, E_D = O.error_decomposition(A, B)
    assert np.allclose(E_T, E_M + E_D, rtol=1e-12)


# ---------------------------------------------------------------- attention
def test_attention_brute_force_tiny():
    rng = np.random.default_rng(2)
    g, n, d = 3, 5, 4
    q, K, V = rng.standard_normal((g, d)), rng.standard_normal((n, d)), rng.standard_normal((n, d))
    out = O.attention(q, K, V)
    for h in range(g):
        w = [math.exp(sum(q[h, c] * K[t, c] for c in range(d)) / math.sqrt(d)) for t in range(n)]
        for c in range(d):
            ref = sum(w[t] * V[t, c] for t in range(n)) / sum(w)
            assert out[h, c] == pytest.approx(ref, rel=1e-12)


def test_attention_matches_torch_sdpa():
    # library routine; residual-only cache => plain SDPA over the raw tokens
    g = torch.Generator().manual_seed(0)
    q = torch.randn(4, 128, generator=g, dtype=torch.float64)
    K = torch.randn(77, 128, generator=g, dtype=torch.float64)
    V = torch.randn(77, 128, generator=g, dtype=torch.float64)
    ref = torch.nn.functional.scaled_dot_product_attention(q[None], K[None], V[None])[0]
    out = O.decode_attention(q.numpy(), [], [], K.numpy(), V.numpy())
    assert np.allclose(out, ref.numpy(), rtol=1e-12, atol=1e-14)


def test_attention_special_cases():
    rng = np.random.default_rng(3)
    V = rng.standard_normal((11, 128))
    # q = 0 => equal logits => mean of V
    assert np.allclose(O.attention(np.zeros((2, 128)), rng.standard_normal((11, 128)), V), V.mean(0))
    # one dominant key => its value
    K = rng.standard_normal((11, 128)); q = 50 * K[4:5]
    assert np.allclose(O.attention(q, K, V), V[4:5], atol=1e-9)
    # empty cache => zeros
    assert np.all(O.attention(np.ones((1, 128)), np.zeros((0, 128)), np.zeros((0, 128))) == 0)
    # rotation invariance of un-quantised attention (online Q/K transforms cancel)
    q = rng.standard_normal((2, 128))
    assert np.allclose(O.attention(O.rotate(q), O.rotate(K), V), O.attention(q, K, V), atol=1e-12)


def test_decode_attention_is_attention_over_dequantised_plus_residual():
    # one chunk + 5 residual tokens, compared with a from-scratch evaluation
    K, V, q, _ = W.config0()
    rng = np.random.default_rng(8)
    kr, vr = rng.standard_normal((5, 128)), rng.standard_normal((5, 128))
    tk, tv = O.quantize_tile(K, "k"), O.quantize_tile(V, "v")
    out = O.decode_attention(q[None], [(tk.codes, tk.s1, tk.s2, tk.z)], [(tv.codes, tv.s1, tv.s2, tv.z)], kr, vr)
    # independent: explicit per-element Eq. 1 + explicit inverse Hadamard by loops on a few rows
    H = scipy.linalg.hadamard(128) / math.sqrt(128)
    Yk = np.empty((128, 128)); Yv = np.empty((128, 128))
    for t in range(128):
        for c in range(128):
            Yk[t, c] = (tk.codes[t, c] + tk.z[c]) * tk.s1[c] * tk.s2[t]     # K: group = channel
            Yv[t, c] = (tv.codes[t, c] + tv.z[t]) * tv.s1[t] * tv.s2[c]     # V: group = token
    Kall = np.vstack([Yk @ H.T, kr]); Vall = np.vstack([Yv @ H.T, vr])
    lg = Kall @ q / math.sqrt(128)
    p = np.exp(lg - lg.max()); p /= p.sum()
    assert np.allclose(out[0], p @ Vall, rtol=1e-11, atol=1e-13)


def test_folded_algebra_equals_plain_definition():
    # The CUDA path never dequantises: it folds H and the scales into q and the
    # output.  This checks that algebra against the
    # oracle's plain definition in float64 (test-side restatement, not oracle code).
    K, V, q, _ = W.config0()
    tk, tv = O.quantize_tile(K, "k"), O.quantize_tile(V, "v")
    ref = O.decode_attention(q[None], [(tk.codes, tk.s1, tk.s2, tk.z)], [(tv.codes, tv.s1, tv.s2, tv.z)],
                             np.zeros((0, 128)), np.zeros((0, 128)))[0]
    H = scipy.linalg.hadamard(128) / math.sqrt(128)
    qr = q.astype(np.float64) @ H
    qt = qr * tk.s1
    beta = (qt * tk.z).sum()
    logit = tk.s2 * (tk.codes.astype(np.float64) @ qt + beta) / math.sqrt(128)
    p = np.exp(logit - logit.max())
    pt = p * tv.s1
    a = pt @ tv.codes.astype(np.float64) + (pt * tv.z).sum()
    out = ((tv.s2 * a) @ H.T) / p.sum()
    assert np.allclose(out, ref, rtol=1e-11, atol=1e-13)


# ---------------------------------------------------------------- three-region layout
def test_cache_partition_brute_force_token_walk():
    # walk the tokens one by one as P:350 describes the regions: the first S go to the sink, later ones
    # trail in FP16 until G of them form a full group, which is then quantised
    for S in (0, 32, 128):
        sink = chunks = trail = 0
        for n in range(0, 700):
            assert O.cache_partition(n, S) == (sink, chunks, trail), (n, S)
            if sink < S:
                sink += 1
            else:
                trail += 1
                if trail == 128:
                    chunks, trail = chunks + 1, 0
    assert O.cache_partition(128 + 3 * 128 + 5, 128) == (128, 3, 5)      # the paper's S = G = 128
    assert O.cache_partition(32 + 128, 32) == (32, 1, 0)                 # IFEval setting S = 32
    assert O.cache_partition(20, 32) == (20, 0, 0)


def test_cache_attention_sink_tokens_are_exact():
    # with every token inside the sink / residual regions nothing is quantised: the result is plain attention
    rng = np.random.default_rng(5)
    K, V, q = rng.standard_normal((150, 128)), rng.standard_normal((150, 128)), rng.standard_normal((2, 128))
    assert np.allclose(O.cache_attention(q, K, V, n_sink=128), O.attention(q, K, V), atol=1e-13)
    # a quantised body changes the result, and the sink region (a x10 first token kept exact) reduces the error
    K2 = rng.standard_normal((128 + 256, 128)); K2[0] *= 10.0
    V2 = rng.standard_normal((128 + 256, 128))
    ref = O.attention(q, K2, V2)
    e_sink = np.abs(O.cache_attention(q, K2, V2, n_sink=128) - ref).max()
    e_none = np.abs(O.cache_attention(q, K2[:384], V2[:384], n_sink=0) - ref).max()
    assert 0 < e_sink < e_none


# ---- multi-token read path (Fig. 4): block_attention ----------------------------------------
def _tiny_cache(rng, n_chunks, r):
    kt, vt = [], []
    for _ in range(n_chunks):
        tk = O.quantize_tile(rng.standard_normal((128, 128)), "k")
        tv = O.quantize_tile(rng.standard_normal((128, 128)), "v")
        kt.append((tk.codes, tk.s1, tk.s2, tk.z)); vt.append((tv.codes, tv.s1, tv.s2, tv.z))
    return kt, vt, rng.standard_normal((r, 128)), rng.standard_normal((r, 128))


def test_block_attention_brute_force_loops():
    """Pin: explicit Python loops over (query token, head, visible token) on a small case."""
    rng = np.random.default_rng(21)
    kt, vt, kr, vr = _tiny_cache(rng, 1, 3)
    n_q, g = 4, 2
    q = rng.standard_normal((n_q, g, 128)); kb = rng.standard_normal((n_q, 128)); vb = rng.standard_normal((n_q, 128))
    out = O.block_attention(q, kt, vt, kr, vr, kb, vb)
    Kc = np.concatenate([O.dequantize_tile(*kt[0], kind="k"), kr]); Vc = np.concatenate([O.dequantize_tile(*vt[0], kind="v"), vr])
    for i in range(n_q):
        for h in range(g):
            keys = [Kc[t] for t in range(len(Kc))] + [kb[t] for t in range(i + 1)]
            vals = [Vc[t] for t in range(len(Vc))] + [vb[t] for t in range(i + 1)]
            lg = [sum(q[i, h, c] * k[c] for c in range(128)) / np.sqrt(128.0) for k in keys]
            m = max(lg); w = [np.exp(x - m) for x in lg]; tot = sum(w)
            ref = sum(wi * v for wi, v in zip(w, vals)) / tot
            assert np.allclose(out[i, h], ref, rtol=1e-10, atol=1e-12)


def test_block_attention_matches_torch_sdpa_causal_mask():
    """Pin: with a raw-only cache the block path is ordinary causal attention with a prefix --
    torch's scaled_dot_product_attention with an explicit boolean mask (library routine)."""
    import torch
    rng = np.random.default_rng(22)
    r, n_q, g = 37, 9, 4
    kr, vr = rng.standard_normal((r, 128)), rng.standard_normal((r, 128))
    q = rng.standard_normal((n_q, g, 128)); kb = rng.standard_normal((n_q, 128)); vb = rng.standard_normal((n_q, 128))
    out = O.block_attention(q, [], [], kr, vr, kb, vb)
    K = torch.tensor(np.concatenate([kr, kb])); V = torch.tensor(np.concatenate([vr, vb]))
    mask = torch.ones((n_q, r + n_q), dtype=torch.bool)
    for i in range(n_q):
        mask[i, r + i + 1:] = False
    qt = torch.tensor(q).permute(1, 0, 2)   # (g, n_q, d)
    ref = torch.nn.functional.scaled_dot_product_attention(qt, K[None].expand(g, -1, -1), V[None].expand(g, -1, -1),
                                                           attn_mask=mask[None]).permute(1, 0, 2).numpy()
    assert np.allclose(out, ref, rtol=1e-10, atol=1e-12)


def test_block_attention_special_cases():
    """n_q = 1 is decode attention with the new token appended to the raw window; the last query of a
    block sees the whole block (no mask); an empty cache leaves query 0 with v_blk[0] exactly."""
    rng = np.random.default_rng(23)
    kt, vt, kr, vr = _tiny_cache(rng, 2, 5)
    g = 4
    q = rng.standard_normal((6, g, 128)); kb = rng.standard_normal((6, 128)); vb = rng.standard_normal((6, 128))
    one = O.block_attention(q[:1], kt, vt, kr, vr, kb[:1], vb[:1])
    assert np.allclose(one[0], O.decode_attention(q[0], kt, vt, np.r_[kr, kb[:1]], np.r_[vr, vb[:1]]), rtol=1e-12)
    out = O.block_attention(q, kt, vt, kr, vr, kb, vb)
    assert np.allclose(out[-1], O.decode_attention(q[-1], kt, vt, np.r_[kr, kb], np.r_[vr, vb]), rtol=1e-12)
    assert np.allclose(out[0], one[0], rtol=1e-12)          # causal: later block tokens do not leak into query 0
    kb2, vb2 = kb.copy(), vb.copy(); kb2[3:] += 100.0; vb2[3:] -= 50.0
    assert np.allclose(O.block_attention(q, kt, vt, kr, vr, kb2, vb2)[:3], out[:3], rtol=1e-12)
    empty = O.block_attention(q, [], [], np.zeros((0, 128)), np.zeros((0, 128)), kb, vb)
    assert np.allclose(empty[0], np.broadcast_to(vb[0], (g, 128)), rtol=1e-12)


# ---- "round-before" aux variant (reading R9b): RTN against the stored FP8 / FP16 parameters ------
def test_rtn_stored_error_is_half_a_stored_step():
    """Pin (error bound): every element whose rounded code is not clipped is reproduced by Eq. 1 WITH THE
    STORED s1 and z to within half a stored step -- the only error left is the rounding to the grid."""
    rng = np.random.default_rng(31)
    for bits, axis in ((2, 1), (4, 1), (2, 0), (4, 0)):
        X = rng.standard_normal((128, 128)) * 3.0 + rng.standard_normal((128, 1))
        ab = np.exp(rng.uniform(-0.3, 2.0, 128))
        codes, s1, z, s1_f, z_f = O.rtn_quantize_stored(X, bits, axis, ab)
        Lv = (1 << bits) - 1
        step = np.expand_dims(s1 / ab, axis)                  # stored step in units of X
        zz = np.expand_dims(z, axis)
        xd = (codes + zz) * step
        raw = X / step - zz
        inside = (raw >= -0.5) & (raw <= Lv + 0.5)
        assert inside.mean() > 0.97                            # FP8 rounds the step by at most 2^-4
        assert np.all(np.abs(xd - X)[inside] <= 0.5 * np.broadcast_to(step, X.shape)[inside] * (1 + 1e-12))
        assert np.all(np.abs(xd - X)[~inside] <= (0.5 + Lv * 2.0 ** -4 + 1e-2) * np.broadcast_to(step, X.shape)[~inside])
        assert np.array_equal(s1, torch.tensor(s1_f).to(torch.float8_e4m3fn).to(torch.float64).numpy())
        assert np.array_equal(z, z_f.astype(np.float16).astype(np.float64))


def test_rtn_stored_equals_plain_rtn_when_parameters_are_representable():
    """Special case: if s * absorbed is an FP8 number and mn / s an FP16 number, rounding first changes nothing."""
    rng = np.random.default_rng(32)
    bits, Lv = 2, 3
    Q = rng.integers(0, Lv + 1, (128, 128)).astype(np.float64)
    Q[:, 0], Q[:, 1] = 0, Lv
    s = 2.0 ** rng.integers(-2, 3, 128).astype(np.float64); z = rng.integers(-8, 8, 128) / 4.0
    X = (Q + z[:, None]) * s[:, None]
    ab = 2.0 ** rng.integers(-1, 2, 128).astype(np.float64)
    c0, s0, z0 = O.rtn_quantize(X, bits, 1)
    c1, s1, z1, _, _ = O.rtn_quantize_stored(X, bits, 1, ab)
    assert np.array_equal(c0, c1) and np.array_equal(c1, Q.astype(np.uint8))
    assert np.array_equal(s1, s0 * ab) and np.array_equal(z1, z0)


def test_round_before_lowers_the_4bit_error():
    """at 4-bit, rounding the aux before RTN removes the FP8 error of the scales from the
    dequantised tile (token-magnitude error ~2.4 % -> ~0.7 %); at 2-bit the two variants are equivalent."""
    K, V = W.kv_tokens(1, 1, 128, seed=33, token_outlier_frac=0.03)
    X = K[0, 0].double().numpy()
    def tokmag(bits, mode, kind):
        t = O.quantize_tile(X, kind, bits=bits, aux_round=mode)
        Xd = O.dequantize_tile(t.codes, t.s1, t.s2, t.z, kind)
        return np.mean(np.abs(np.linalg.norm(Xd, axis=1) / np.linalg.norm(X, axis=1) - 1))
    for kind in "kv":
        assert tokmag(4, "before", kind) < 0.5 * tokmag(4, "after", kind)
        assert abs(tokmag(2, "before", kind) / tokmag(2, "after", kind) - 1) < 0.3


# ---- Hadamard arrangement (App. A): online q / K transform after RoPE, absorbed W_V / W_O ----
def _rope_table(pos, d=128, base=10000.0):
    inv = base ** (-np.arange(0, d, 2) / d)
    ang = np.asarray(pos, dtype=np.float64)[:, None] * inv[None, :]
    return np.cos(ang), np.sin(ang)


def test_rope_is_a_complex_rotation_and_relative():
    """Pin: the half-split RoPE is multiplication of z_c = x[c] + i x[c + d/2] by e^{i angle_c} (textbook form),
    preserves norms, and q(m) . k(n) depends only on m - n."""
    rng = np.random.default_rng(41)
    x = rng.standard_normal((5, 128)); pos = np.array([0, 1, 7, 100, 4095])
    cos, sin = _rope_table(pos)
    y = O.rope_rotate_half(x, cos, sin)
    zc = (x[:, :64] + 1j * x[:, 64:]) * (cos + 1j * sin)
    assert np.allclose(y[:, :64], zc.real, atol=1e-12) and np.allclose(y[:, 64:], zc.imag, atol=1e-12)
    assert np.allclose(np.linalg.norm(y, axis=1), np.linalg.norm(x, axis=1))
    q, k = rng.standard_normal(128), rng.standard_normal(128)
    def dot(m, n):
        cm, sm_ = _rope_table([m]); cn, sn = _rope_table([n])
        return float(O.rope_rotate_half(q[None], cm, sm_)[0] @ O.rope_rotate_half(k[None], cn, sn)[0])
    assert np.isclose(dot(10, 3), dot(1010, 1003)) and not np.isclose(dot(10, 3), dot(10, 4))


def test_rope_hadamard_preserves_attention_logits():
    rng = np.random.default_rng(42)
    q, k = rng.standard_normal((3, 128)), rng.standard_normal((9, 128))
    cq, sq = _rope_table([20, 21, 22]); ck, sk = _rope_table(np.arange(9))
    plain = O.rope_rotate_half(q, cq, sq) @ O.rope_rotate_half(k, ck, sk).T
    assert np.allclose(O.rope_hadamard(q, cq, sq) @ O.rope_hadamard(k, ck, sk).T, plain, atol=1e-10)


def test_absorbed_hadamards_cancel():
    """the transforms merged into W_V and W_O leave the layer's function unchanged:
    softmax(.) (x W_V') W_O' = softmax(.) (x W_V) W_O for any attention weights (GQA: Hq = 2 Hkv here)."""
    rng = np.random.default_rng(43)
    dm, Hkv, Hq = 48, 2, 4
    W_V, W_O = rng.standard_normal((dm, Hkv * 128)), rng.standard_normal((Hq * 128, dm))
    Wv2, Wo2 = O.absorb_hadamard(W_V, W_O)
    x = rng.standard_normal((7, dm)); P_ = rng.random((Hq, 7)); P_ /= P_.sum(1, keepdims=True)
    def layer(Wv, Wo):
        v = (x @ Wv).reshape(7, Hkv, 128)
        a = np.concatenate([P_[h] @ v[:, h // 2] for h in range(Hq)])      # (Hq * 128,)
        return a @ Wo
    assert np.allclose(layer(Wv2, Wo2), layer(W_V, W_O), atol=1e-9)
    assert np.allclose((x @ Wv2).reshape(7, Hkv, 128), O.rotate((x @ W_V).reshape(7, Hkv, 128)), atol=1e-10)
