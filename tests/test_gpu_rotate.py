"""GPU parity: the Hadamard arrangement kernels (App. A) through the C ABI vs the
oracle's rope_hadamard / absorb_hadamard, and the pre-rotated cache route (rotate_k = rotate_v = 0)."""
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


def _rope_table(pos, base=10000.0):
    inv = base ** (-np.arange(0, 128, 2) / 128.0)
    ang = np.asarray(pos, dtype=np.float64)[:, None] * inv[None, :]
    return np.cos(ang), np.sin(ang)


def _rand(shape, seed, dtype):
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    return torch.randn(shape, generator=g, device="cuda").to(dtype)


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
@pytest.mark.parametrize("n_tok,n_heads", [(1, 1), (37, 5), (300, 32)])
def test_rope_hadamard_vs_oracle(kv, dtype, n_tok, n_heads):
    x = _rand((n_tok, n_heads, 128), 7 + n_tok, dtype)
    cos, sin = _rope_table(np.arange(n_tok) * 17 % 4099)
    ct, st = (torch.tensor(a, dtype=torch.float32, device="cuda") for a in (cos, sin))
    # the kernel sees the fp32-rounded table: the oracle gets the same values
    c64, s64 = ct.double().cpu().numpy()[:, None, :], st.double().cpu().numpy()[:, None, :]
    tol = 2e-6 if dtype == torch.float32 else 2 ** -8
    for rotate in (True, False):
        y = kv.rope_hadamard(x, ct, st, rotate=rotate).double().cpu().numpy()
        ref = O.rope_hadamard(P.tile_f64(x), c64, s64) if rotate else O.rope_rotate_half(P.tile_f64(x), c64, s64)
        assert np.abs(y - ref).max() <= tol * np.abs(ref).max(), np.abs(y - ref).max()
    y = kv.rope_hadamard(x).double().cpu().numpy()                   # no RoPE: plain head-wise rotation
    ref = O.rotate(P.tile_f64(x))
    assert np.abs(y - ref).max() <= tol * np.abs(ref).max()


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16])
def test_absorbed_transforms_vs_oracle(kv, dtype):
    dm, Hkv, Hq = 200, 2, 4                                            # d_model not a multiple of 32: ragged column tail
    W_V, W_O = _rand((dm, Hkv * 128), 11, dtype), _rand((Hq * 128, dm), 12, dtype)
    Wv_ref, Wo_ref = O.absorb_hadamard(P.tile_f64(W_V), P.tile_f64(W_O))
    Wv, Wo = kv.hadamard_rows(W_V).double().cpu().numpy(), kv.hadamard_row_groups(W_O).double().cpu().numpy()
    tol = 2e-6 if dtype == torch.float32 else 2 ** -8
    assert np.abs(Wv - Wv_ref).max() <= tol * np.abs(Wv_ref).max()
    assert np.abs(Wo - Wo_ref).max() <= tol * np.abs(Wo_ref).max()
    # in place
    w2 = W_O.clone(); kv.hadamard_row_groups(w2, out=w2)
    assert torch.equal(w2.double().cpu(), torch.tensor(Wo))
    # applying the (symmetric, orthonormal) rotation twice gives the input back
    if dtype == torch.float32:
        back = kv.hadamard_rows(kv.hadamard_rows(W_V))
        assert (back - W_V).abs().max().item() <= 1e-5 * W_V.abs().max().item()


def test_prerotated_cache_route_equals_online_rotation(kv):
    """q, K rotated by kvarn_rope_hadamard and V by the absorbed W_V transform, cache written and read with
    rotate_k = rotate_v = 0: the rotated-space output times R^T equals the standard route's output (fp32 inputs)."""
    B, Hq, Hkv, n_tok = 2, 8, 2, 128 * 3 + 50
    K, V = W.kv_tokens(B, Hkv, n_tok, seed=51, device="cuda", dtype=torch.float32)
    q = W.queries(B, Hq, seed=51, device="cuda", dtype=torch.float32)
    p1 = kv.default_params(2)
    c1 = kv.Cache(p1, B, Hkv, 4, resid_dtype=torch.float32); kv.prefill(p1, c1, K, V)
    out1 = kv.decode_attention(p1, c1, q)
    Kr = kv.rope_hadamard(K.reshape(-1, 1, 128)).reshape(K.shape)     # positions already applied upstream: rotation only
    Vr = kv.hadamard_rows(V)
    qr = kv.rope_hadamard(q.reshape(-1, 1, 128)).reshape(q.shape)
    p0 = kv.default_params(2, rotate_k=0, rotate_v=0)
    c0 = kv.Cache(p0, B, Hkv, 4, resid_dtype=torch.float32); kv.prefill(p0, c0, Kr, Vr)
    out0 = kv.decode_attention(p0, c0, qr)                               # in the rotated space
    back = kv.hadamard_rows(out0)                                        # R^T = R
    err = (back - out1).abs().amax(dim=-1) / out1.abs().amax(dim=-1)
    assert err.max().item() <= P.ATTN_RTOL, err.max().item()


def test_rotate_argument_checks(kv):
    x = torch.zeros((4, 2, 128), dtype=torch.float32, device="cuda")
    assert kv.rope_hadamard(x[:0].contiguous()).shape[0] == 0
    w = torch.zeros((100, 8), dtype=torch.float32, device="cuda")       # rows not a multiple of 128
    with pytest.raises(kv.KvarnError, match="INVALID_ARG"):
        kv.hadamard_row_groups(w)
