"""KVarN CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A plain, slow, float64 numpy restatement of what the KVarN hot path computes,
written from /root/reference/PAPER.md (cited below as ``P:<line>``) and the
readings of its silent / garbled points listed in DESIGN.md ("Readings").

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this module.  It shares no code with the
CUDA path under ``paper_2606_03458_b200/`` and imports nothing from it.

What is here
------------
* the quantizer, **step by step in the paper's order** (it is an encoding):
  Hadamard rotation (Fig. 2, Sec. 2.2, Sec. 3.3, App. A)
  -> VarN, Algorithm 1 verbatim -> asymmetric round-to-nearest,
  K per channel / V per token (Sec. 2.1, Eq. 1) -> auxiliary storage,
  two FP8 scales + one FP16 zero-point per 128 elements;
* dual-scale dequantisation, Eq. 1 plus the second scale;
* attention over the dequantised cache and the raw residual window, as the
  **plain definition** softmax(q K^T / sqrt(d)) V (P:9).

Pin status (tests/test_oracle_*.py, ``-m "not gpu"``)
-----------------------------------------------------
hadamard / rotate ........ pinned (H H^T = d I, scipy.linalg.hadamard, norms)
varn ..................... pinned (closed form E*diag(b), clamp case, invariants)
imbalance ................ pinned to its stated formula only -- the body of
                           IMB() is lost in PAPER.md; the formula
                           is reading R1 in DESIGN.md, a reconstruction
rtn_quantize / dequant ... pinned (on-grid round trip, textbook min-max RTN)
fp8 / fp16 rounding ...... pinned (torch.float8_e4m3fn, numpy.float16 casts)
attention ................ pinned (brute-force loops, torch SDPA, invariances)
cache_partition .......... pinned (brute-force token walk, P:350's S/G/R settings)
block_attention .......... pinned (brute-force loops, torch SDPA with a causal mask,
                           n_q = 1 and last-query special cases)
rope_hadamard / absorb_hadamard ... pinned (complex-number form of RoPE, relative-position
                           invariance, q.k and a W_O preserved by the rotations)
codes / scales of a tile vs values printed by the paper ... **parity unpinned**:
                           the paper prints no intermediate value for any tile.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

HEAD_DIM = 128
CHUNK = 128

# Algorithm 1 constants.  The log clamps are the paper's; the
# variance limits c_min / c_max are inputs the paper leaves without values
# -> reading R2; K = 8 is the iteration count of Sec. 4.2 -> R3.
VARN_ITERS = 8
VARN_LOG_LO = -0.3
VARN_LOG_HI = 10.0
VARN_C_MIN = 1e-8
VARN_C_MAX = 1e8

# RTN: a group whose range is below this is "degenerate" (reading R7).
RTN_DEGENERATE = 1e-12


# --------------------------------------------------------------------------
# Hadamard rotation
# --------------------------------------------------------------------------
def hadamard_matrix(d: int = HEAD_DIM) -> np.ndarray:
    """Sylvester Walsh-Hadamard matrix H_d (entries +-1, natural order).

    H_1 = [1];  H_2n = [[H_n, H_n], [H_n, -H_n]].  No random sign diagonal
    (reading R6).  Built explicitly -- the oracle has no butterfly code.
    """
    if d < 1 or d & (d - 1):
        raise ValueError("d must be a power of two")
    H = np.ones((1, 1), dtype=np.float64)
    while H.shape[0] < d:
        H = np.block([[H, H], [H, -H]])
    return H


def rotate(X: np.ndarray) -> np.ndarray:
    """Y[t, :] = X[t, :] @ H_d / sqrt(d): every token rotated along channels.

    "Every token is Hadamard-rotated in the channel dimension".  The
    orthonormal scaling makes it a rotation; H/sqrt(d) is symmetric and
    its own inverse, so ``rotate(rotate(X)) == X``.
    """
    X = np.asarray(X, dtype=np.float64)
    d = X.shape[-1]
    return X @ (hadamard_matrix(d) / np.sqrt(d))


# --------------------------------------------------------------------------
# VarN -- Algorithm 1
# --------------------------------------------------------------------------
def _var(C: np.ndarray, axis: int) -> np.ndarray:
    """Population variance (divide by n), mean-centred -- reading R4."""
    m = C.mean(axis=axis, keepdims=True)
    return ((C - m) ** 2).mean(axis=axis)


def imbalance(C: np.ndarray, c_min: float = VARN_C_MIN) -> float:
    """IMB(X) of Alg. 1 -- body lost in the PDF extraction.

    Reading R1 (a reconstruction, not paper text): with "variances across
    dims 2 and 1" (the one surviving comment) pooled,
        Imb = max(all row and column variances) / max(min(same), c_min).
    """
    v = np.concatenate([_var(C, axis=1), _var(C, axis=0)])
    return float(v.max() / max(v.min(), c_min))


@dataclass
class VarNResult:
    T_bal: np.ndarray          # (R, C) balanced tile  T / S_c* / S_r*
    S_c: np.ndarray            # (C,) best column scales  exp(L_c)
    S_r: np.ndarray            # (R,) best row scales     exp(L_r)
    k_best: int                # iterate the "<=" rule kept (0 = initial)
    # whole trajectory, index k = 0..K (0 = before the first iteration)
    I: list = field(default_factory=list)
    S_c_k: list = field(default_factory=list)
    S_r_k: list = field(default_factory=list)


def varn(T: np.ndarray, iters: int = VARN_ITERS, c_min: float = VARN_C_MIN,
         c_max: float = VARN_C_MAX, log_lo: float = VARN_LOG_LO,
         log_hi: float = VARN_LOG_HI) -> VarNResult:
    """Algorithm 1, one tile (N = 1), in the paper's order and notation.

    ``T`` is (R, C).  Line numbers are Alg. 1's.
    """
    T = np.asarray(T, dtype=np.float64)
    R, Cn = T.shape
    L_c = np.zeros((1, Cn))                                   # line 5
    L_r = np.zeros((R, 1))
    C = (T / np.exp(L_c)) / np.exp(L_r)                       # line 6
    I_best = imbalance(C, c_min)                              # line 7
    S_c_best, S_r_best = np.exp(L_c), np.exp(L_r)             # line 8
    k_best = 0
    res = VarNResult(None, None, None, 0)
    res.I.append(I_best)
    res.S_c_k.append(S_c_best.ravel().copy())
    res.S_r_k.append(S_r_best.ravel().copy())
    for k in range(1, iters + 1):                             # line 9
        # line 10: Var_row = variance taken ALONG the row index (over the R
        # rows), one value per column -- it feeds the 1 x C vector L_c.
        v_col = np.clip(_var(C, axis=0), c_min, c_max)[None, :]
        L_c = np.clip(L_c + 0.5 * np.log(v_col), log_lo, log_hi)   # line 11
        C = (T / np.exp(L_c)) / np.exp(L_r)                   # line 12
        v_row = np.clip(_var(C, axis=1), c_min, c_max)[:, None]    # line 13
        L_r = np.clip(L_r + 0.5 * np.log(v_row), log_lo, log_hi)   # line 14
        C = (T / np.exp(L_c)) / np.exp(L_r)                   # line 15
        I_curr = imbalance(C, c_min)                          # line 16
        res.I.append(I_curr)
        res.S_c_k.append(np.exp(L_c).ravel().copy())
        res.S_r_k.append(np.exp(L_r).ravel().copy())
        if I_curr <= I_best:                                  # line 18
            I_best = I_curr                                   # line 19
            S_c_best, S_r_best = np.exp(L_c), np.exp(L_r)     # line 20
            k_best = k
    res.T_bal = (T / S_c_best) / S_r_best                     # line 24
    res.S_c = S_c_best.ravel().copy()
    res.S_r = S_r_best.ravel().copy()
    res.k_best = k_best
    return res


def varn_at(T: np.ndarray, traj: VarNResult, k: int):
    """Balanced tile and scales of iterate ``k`` of a trajectory (reading R10:
    several iterates are "correct"; the harness compares at the GPU's k)."""
    S_c, S_r = traj.S_c_k[k], traj.S_r_k[k]
    T = np.asarray(T, dtype=np.float64)
    return (T / S_c[None, :]) / S_r[:, None], S_c, S_r


# --------------------------------------------------------------------------
# Asymmetric round-to-nearest (Eq. 1)
# --------------------------------------------------------------------------
def rtn_quantize(X: np.ndarray, bits: int, group_axis: int):
    """Asymmetric RTN with one (scale, zero) per group.

    ``group_axis`` is the axis a group runs ALONG (its 128 members).  Returns
    (codes uint8 same shape as X, s, z) with s, z indexed by the other axis,
    such that Eq. 1 holds:  X_dq = (codes + z) * s
    Reading R7: s = (mx - mn) / Lv, z = mn / s (a real number in code units),
    codes = clip(rint(x / s - z), 0, Lv) with rint = half-to-even; a group with
    mx - mn < 1e-12 gets s = 1, codes = 0, z = mn.
    """
    X = np.asarray(X, dtype=np.float64)
    Lv = (1 << bits) - 1
    mn = X.min(axis=group_axis, keepdims=True)
    mx = X.max(axis=group_axis, keepdims=True)
    rng = mx - mn
    degenerate = rng < RTN_DEGENERATE
    s = np.where(degenerate, 1.0, rng / Lv)
    z = mn / s
    codes = np.clip(np.rint(X / s - z), 0, Lv)
    codes = np.where(degenerate, 0.0, codes).astype(np.uint8)
    return codes, np.squeeze(s, axis=group_axis), np.squeeze(z, axis=group_axis)


def rtn_dequantize(codes: np.ndarray, s: np.ndarray, z: np.ndarray,
                   group_axis: int) -> np.ndarray:
    """Eq. 1:  X_dq = (X_q + z) (.) s."""
    s = np.expand_dims(np.asarray(s, dtype=np.float64), group_axis)
    z = np.expand_dims(np.asarray(z, dtype=np.float64), group_axis)
    return (codes.astype(np.float64) + z) * s


# --------------------------------------------------------------------------
# Auxiliary storage formats: FP8 scales, FP16 zero-point
# --------------------------------------------------------------------------
def round_fp8_e4m3(x: np.ndarray) -> np.ndarray:
    """Round to the nearest FP8 E4M3 ("fn": finite, max 448) value, ties to
    even, saturating at +-448 (reading R9).  Returns float64 values.

    E4M3: 1 sign, 4 exponent (bias 7), 3 mantissa bits; subnormal step 2^-9;
    normal binade 2^e has step 2^(e-3) for e in [-6, 8].
    """
    x = np.asarray(x, dtype=np.float64)
    a = np.abs(x)
    e = np.floor(np.log2(np.maximum(a, 2.0 ** -20)))
    e = np.clip(e, -6, 8)
    step = 2.0 ** (e - 3)
    r = np.rint(a / step) * step          # rint = half-to-even on the grid
    r = np.minimum(r, 448.0)
    return np.sign(x) * r


def fp8_e4m3_bits(x: np.ndarray) -> np.ndarray:
    """Byte encoding of values already on the E4M3 grid (non-negative or not)."""
    x = np.asarray(x, dtype=np.float64)
    a = np.abs(x)
    sign = (np.signbit(x)).astype(np.uint8) << 7
    e = np.floor(np.log2(np.maximum(a, 2.0 ** -20)))
    sub = a < 2.0 ** -6
    e = np.clip(e, -6, 8)
    mant_sub = np.rint(a / 2.0 ** -9)
    mant_norm = np.rint(a / 2.0 ** (e - 3)) - 8
    bits = np.where(sub, mant_sub, ((e + 7) * 8 + mant_norm)).astype(np.uint8)
    return (bits | sign).astype(np.uint8)


def fp8_e4m3_from_bits(b: np.ndarray) -> np.ndarray:
    b = np.asarray(b, dtype=np.uint8).astype(np.int64)
    sign = np.where(b & 0x80, -1.0, 1.0)
    e = (b >> 3) & 0xF
    m = b & 7
    val = np.where(e == 0, m * 2.0 ** -9, (8 + m) * 2.0 ** (e.astype(np.float64) - 10))
    return sign * val


def round_fp16(x: np.ndarray) -> np.ndarray:
    """Round to IEEE binary16 (ties to even); numpy's cast is the definition."""
    with np.errstate(over="ignore"):
        return np.asarray(x, dtype=np.float64).astype(np.float16).astype(np.float64)


# --------------------------------------------------------------------------
# One tile through the whole write path (Fig. 2)
# --------------------------------------------------------------------------
@dataclass
class QuantTile:
    """What is stored for one (head_dim x token-chunk) tile.

    codes[t, c] in 0..2^bits-1.  ``s1``/``z`` are indexed by the RTN group
    (K: channel c, V: token t), ``s2`` by the other axis (K: token, V: channel).
    ``*_f`` are the pre-storage (unrounded) values; the un-suffixed ones are
    what is stored (FP8 / FP8 / FP16), as float64.
    """
    kind: str
    bits: int
    codes: np.ndarray
    s1: np.ndarray
    s2: np.ndarray
    z: np.ndarray
    s1_f: np.ndarray
    s2_f: np.ndarray
    z_f: np.ndarray
    k_best: int
    varn: VarNResult


def rtn_quantize_stored(X: np.ndarray, bits: int, group_axis: int, absorbed: np.ndarray):
    """RTN against the STORED parameters ("round-before", reading R9b; P:382 stores s1 as FP8 and z as FP16,
    the paper does not say whether the codes are taken before or after that rounding).

    Per group: mn, mx, s = (mx - mn) / Lv as in ``rtn_quantize``; the scale that will be stored is
    s1 = fp8(s * absorbed) (``absorbed`` = the Sinkhorn scale constant along the group, R8), so the step the
    dequantiser really applies, in units of X, is s' = s1 / absorbed; z = fp16(mn / s');
    codes = clip(rint(x / s' - z), 0, Lv).  A group whose s1 rounds to zero keeps s' = s.
    Returns (codes, s1 (stored), z (stored), s1_f = s * absorbed, z_f = mn / s')."""
    X = np.asarray(X, dtype=np.float64)
    Lv = (1 << bits) - 1
    ab = np.expand_dims(np.asarray(absorbed, dtype=np.float64), group_axis)
    mn = X.min(axis=group_axis, keepdims=True)
    mx = X.max(axis=group_axis, keepdims=True)
    rng = mx - mn
    degenerate = rng < RTN_DEGENERATE
    s = np.where(degenerate, 1.0, rng / Lv)
    s1_f = s * ab
    s1 = round_fp8_e4m3(s1_f)
    s_used = np.where(s1 > 0, s1 / ab, s)
    z_f = mn / s_used
    z = round_fp16(z_f)
    codes = np.clip(np.rint(X / s_used - z), 0, Lv)
    codes = np.where(degenerate, 0.0, codes).astype(np.uint8)
    sq = lambda a: np.squeeze(a, axis=group_axis)
    return codes, sq(s1), sq(z), sq(s1_f), sq(z_f)


def quantize_tile(X: np.ndarray, kind: str, bits: int = 2, iters: int = VARN_ITERS,
                  rotate_on: bool = True, at_k: int | None = None,
                  c_min: float = VARN_C_MIN, c_max: float = VARN_C_MAX,
                  aux_round: str = "after") -> QuantTile:
    """Hadamard -> VarN -> RTN -> aux rounding, for one tile X[t, c] (128 x 128).

    kind 'k': RTN groups are channels (each over the chunk's tokens);
    kind 'v': RTN groups are tokens (each over the channels).
    ``at_k`` forces the iterate used (reading R10); default = Alg. 1's choice.
    ``aux_round``: "after" (default, reading R9: codes from the unrounded parameters, aux rounded for
    storage afterwards) or "before" (R9b: the second scale is rounded to FP8 first, the tile is balanced
    with the rounded value, and RTN runs against the stored s1 / z -- ``rtn_quantize_stored``).
    """
    assert kind in ("k", "v")
    X = np.asarray(X, dtype=np.float64)
    Y = rotate(X) if rotate_on else X                      # step 1
    # step 2: the base tile is (head-dim x token-chunk): rows R =
    # channels, columns C = tokens (reading R5) => S_c per token, S_r per channel.
    T = Y.T
    vr = varn(T, iters=iters, c_min=c_min, c_max=c_max)
    if at_k is None:
        T_bal, S_c, S_r, k = vr.T_bal, vr.S_c, vr.S_r, vr.k_best
    else:
        T_bal, S_c, S_r = varn_at(T, vr, at_k)
        k = at_k
    if aux_round == "before":
        if kind == "k":      # second scale = S_c (per token), absorbed = S_r (per channel)
            s2 = round_fp8_e4m3(S_c)
            codes_ct, s1, z, s1_f, z_f = rtn_quantize_stored(T / s2[None, :] / S_r[:, None], bits, 1, S_r)
            s2_f = S_c
        else:                # second scale = S_r (per channel), absorbed = S_c (per token)
            s2 = round_fp8_e4m3(S_r)
            codes_ct, s1, z, s1_f, z_f = rtn_quantize_stored(T / S_c[None, :] / s2[:, None], bits, 0, S_c)
            s2_f = S_r
        return QuantTile(kind=kind, bits=bits, codes=np.ascontiguousarray(codes_ct.T), s1=s1, s2=s2, z=z,
                         s1_f=s1_f, s2_f=s2_f, z_f=z_f, k_best=k, varn=vr)
    assert aux_round == "after"
    # step 3: RTN on the balanced tile.  T_bal is [channel, token].
    if kind == "k":      # per channel: group runs along tokens (axis 1)
        codes_ct, s, z = rtn_quantize(T_bal, bits, group_axis=1)
        s1_f, s2_f = s * S_r, S_c            # step 4 (reading R8)
    else:                # per token: group runs along channels (axis 0)
        codes_ct, s, z = rtn_quantize(T_bal, bits, group_axis=0)
        s1_f, s2_f = s * S_c, S_r
    return QuantTile(kind=kind, bits=bits, codes=np.ascontiguousarray(codes_ct.T),
                     s1=round_fp8_e4m3(s1_f), s2=round_fp8_e4m3(s2_f), z=round_fp16(z),
                     s1_f=s1_f, s2_f=s2_f, z_f=z, k_best=k, varn=vr)


def dequantize_tile(codes: np.ndarray, s1: np.ndarray, s2: np.ndarray, z: np.ndarray,
                    kind: str, rotate_on: bool = True) -> np.ndarray:
    """Eq. 1 with the second scale, then the inverse rotation.

    Yhat[t, c] = (codes[t, c] + z_g) * s1_g * s2_o,  g = RTN group index,
    o = the other axis;  X_dq = Yhat @ H^T / sqrt(d).
    """
    q = np.asarray(codes, dtype=np.float64)                # [t, c]
    if kind == "k":      # group = channel c, other = token t
        Yhat = (q + z[None, :]) * s1[None, :] * s2[:, None]
    else:                # group = token t, other = channel c
        Yhat = (q + z[:, None]) * s1[:, None] * s2[None, :]
    if not rotate_on:
        return Yhat
    d = Yhat.shape[-1]
    return Yhat @ (hadamard_matrix(d).T / np.sqrt(d))


# --------------------------------------------------------------------------
# Attention: the plain definition (P:9; residual window P:350)
# --------------------------------------------------------------------------
def attention(q: np.ndarray, K: np.ndarray, V: np.ndarray, sm_scale: float | None = None
              ) -> np.ndarray:
    """softmax(q K^T * sm_scale) V for one KV head.

    q: (g, d) query heads sharing the KV head; K, V: (n, d).  float64.
    """
    q = np.asarray(q, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    V = np.asarray(V, dtype=np.float64)
    if sm_scale is None:
        sm_scale = 1.0 / np.sqrt(q.shape[-1])
    if K.shape[0] == 0:
        return np.zeros((q.shape[0], V.shape[-1]))
    logits = (q @ K.T) * sm_scale
    logits = logits - logits.max(axis=-1, keepdims=True)
    p = np.exp(logits)
    p = p / p.sum(axis=-1, keepdims=True)
    return p @ V


def decode_attention(q: np.ndarray, k_tiles: list, v_tiles: list,
                     k_resid: np.ndarray, v_resid: np.ndarray,
                     sm_scale: float | None = None, rotate_k: bool = True,
                     rotate_v: bool = True) -> np.ndarray:
    """Attention of (g, d) queries over [dequantised chunks ; raw residual].

    ``k_tiles`` / ``v_tiles``: lists of (codes, s1, s2, z) with the STORED aux
    values (step 5 of the oracle), one per 128-token chunk, oldest first.
    ``k_resid`` / ``v_resid``: (r, d) raw tokens not yet quantised.
    """
    d = np.asarray(q).shape[-1]
    Ks = [dequantize_tile(*t, kind="k", rotate_on=rotate_k) for t in k_tiles]
    Vs = [dequantize_tile(*t, kind="v", rotate_on=rotate_v) for t in v_tiles]
    Ks.append(np.asarray(k_resid, dtype=np.float64).reshape(-1, d))
    Vs.append(np.asarray(v_resid, dtype=np.float64).reshape(-1, d))
    return attention(q, np.concatenate(Ks, axis=0), np.concatenate(Vs, axis=0), sm_scale)


# --------------------------------------------------------------------------
# Three-region cache layout (App. D "Quantization")
# --------------------------------------------------------------------------
def cache_partition(n_tok: int, n_sink: int = 0, group: int = 128):
    """(sink, chunks, residual) of a sequence of ``n_tok`` tokens: "S sink tokens in
    FP16 ..., a 2-bit quantized body composed of groups of G tokens each, and R trailing tokens
    in FP16 ... which have not yet accumulated enough context to form a full quantization group".
    The first min(n_tok, S) tokens are the sink, every complete group of G after them is
    quantised, the rest trail in FP16 (reading R11: quantised the moment a group is complete)."""
    sink = min(n_tok, n_sink)
    body = n_tok - sink
    return sink, body // group, body % group


def cache_attention(q: np.ndarray, K: np.ndarray, V: np.ndarray, n_sink: int = 0, bits: int = 2,
                    sm_scale: float | None = None) -> np.ndarray:
    """End-to-end definition for one KV head: partition the (n_tok, d) raw K, V by
    ``cache_partition``, quantise the body chunk by chunk (steps 1-4), and attend over
    [raw sink ; dequantised body ; raw residual] (steps 5-6)."""
    K = np.asarray(K, dtype=np.float64); V = np.asarray(V, dtype=np.float64)
    ns, nc, r = cache_partition(K.shape[0], n_sink)
    kt, vt = [], []
    for c in range(nc):
        sl = slice(ns + 128 * c, ns + 128 * (c + 1))
        tk, tv = quantize_tile(K[sl], "k", bits=bits), quantize_tile(V[sl], "v", bits=bits)
        kt.append((tk.codes, tk.s1, tk.s2, tk.z)); vt.append((tv.codes, tv.s1, tv.s2, tv.z))
    raw = np.r_[0:ns, ns + 128 * nc:K.shape[0]]
    return decode_attention(q, kt, vt, K[raw], V[raw], sm_scale=sm_scale)


# --------------------------------------------------------------------------
# Multi-token read path: a block of new tokens against the compressed cache
# (Fig. 4 "pseudo-decode", Sec. 3.2)
# --------------------------------------------------------------------------
def block_attention(q_blk: np.ndarray, k_tiles: list, v_tiles: list,
                    k_raw: np.ndarray, v_raw: np.ndarray,
                    k_blk: np.ndarray, v_blk: np.ndarray,
                    sm_scale: float | None = None) -> np.ndarray:
    """Causal attention of a block of ``n_q`` new tokens for one KV head (Fig. 4: "We split
    the sequence into blocks of size b. After every block, the freshly produced K, V are quantized
    before being written back to the KV-cache. Subsequent blocks access a *quantized* cache").

    Query i of the block sees every token of the cache -- dequantised chunks ``k_tiles`` /
    ``v_tiles`` (stored aux, as in ``decode_attention``) and the raw sink / residual tokens
    ``k_raw`` / ``v_raw`` (r, d) -- plus the block's own, not yet quantised tokens 0..i
    (``k_blk`` / ``v_blk`` (n_q, d)).  Plain definition, one query token at a time.

    q_blk: (n_q, g, d).  Returns (n_q, g, d) float64.
    """
    q_blk = np.asarray(q_blk, dtype=np.float64)
    k_blk = np.asarray(k_blk, dtype=np.float64)
    v_blk = np.asarray(v_blk, dtype=np.float64)
    n_q, _, d = q_blk.shape
    k_raw = np.asarray(k_raw, dtype=np.float64).reshape(-1, d)
    v_raw = np.asarray(v_raw, dtype=np.float64).reshape(-1, d)
    out = np.zeros_like(q_blk)
    for i in range(n_q):
        out[i] = decode_attention(q_blk[i], k_tiles, v_tiles,
                                  np.concatenate([k_raw, k_blk[:i + 1]], axis=0),
                                  np.concatenate([v_raw, v_blk[:i + 1]], axis=0), sm_scale=sm_scale)
    return out


# --------------------------------------------------------------------------
# Hadamard arrangement around the attention layer (App. A, Fig. 7)
# --------------------------------------------------------------------------
def rope_rotate_half(x: np.ndarray, cos: np.ndarray, sin: np.ndarray) -> np.ndarray:
    """Rotary embedding in the half-split convention of the Llama / Qwen models the paper evaluates:
    channel c < d/2 is paired with c + d/2;  y[c] = x[c] cos[c] - x[c+d/2] sin[c],
    y[c+d/2] = x[c+d/2] cos[c] + x[c] sin[c].  x: (..., d); cos, sin: (..., d/2) broadcastable.
    The paper only says the online transforms come "after the RoPE-embedding"; the caller
    supplies the cos / sin table, so no frequency base is fixed here."""
    x = np.asarray(x, dtype=np.float64)
    h = x.shape[-1] // 2
    x1, x2 = x[..., :h], x[..., h:]
    return np.concatenate([x1 * cos - x2 * sin, x2 * cos + x1 * sin], axis=-1)


def rope_hadamard(x: np.ndarray, cos: np.ndarray, sin: np.ndarray) -> np.ndarray:
    """The online transform of q and K ("two online transforms after the RoPE-embedding ...
    head-wise"): y = RoPE(x) H / sqrt(d) per head.  x: (..., d)."""
    return rotate(rope_rotate_half(x, cos, sin))


def absorb_hadamard(W_V: np.ndarray, W_O: np.ndarray, d: int = HEAD_DIM):
    """The two absorbed transforms ("merged with W_V and W_O respectively and do not need to be
    computed during inference").  With v = x W_V (W_V: (d_model, Hkv d)) and out = a W_O
    (W_O: (Hq d, d_model)), block-diagonal R = diag(H / sqrt(d)):  W_V' = W_V R,  W_O' = R^T W_O, so that
    v' = v R per head is what gets quantised (rotate_v = 0 at run time) and a' W_O' = a W_O."""
    W_V = np.asarray(W_V, dtype=np.float64); W_O = np.asarray(W_O, dtype=np.float64)
    R = hadamard_matrix(d) / np.sqrt(d)
    Wv = W_V.reshape(W_V.shape[0], -1, d) @ R
    Wo = np.einsum("ij,hjm->him", R.T, W_O.reshape(-1, d, W_O.shape[1]))
    return Wv.reshape(W_V.shape), Wo.reshape(W_O.shape)


# --------------------------------------------------------------------------
# Diagnostics (oracle side only): Eq. 2-3 error decomposition
# --------------------------------------------------------------------------
def error_decomposition(K: np.ndarray, K_dq: np.ndarray):
    """Per-token E_T = E_M + E_D (Eq. 3)."""
    K = np.asarray(K, dtype=np.float64)
    K_dq = np.asarray(K_dq, dtype=np.float64)
    nk = np.linalg.norm(K, axis=-1)
    nd = np.linalg.norm(K_dq, axis=-1)
    cos = (K * K_dq).sum(-1) / np.maximum(nk * nd, 1e-300)
    E_T = ((K - K_dq) ** 2).sum(-1)
    E_M = (nk - nd) ** 2
    E_D = 2 * nk * nd * (1 - cos)
    return E_T, E_M, E_D
