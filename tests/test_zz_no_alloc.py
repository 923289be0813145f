"""GPU: kvarn_decode_attention_static (the read path with its split-K scratch in the library's static device array --
for callers that cannot call cudaMalloc) against kvarn_decode_attention with a caller-owned workspace.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests.
The static array is shared by every call and keeps the last call's contents, so the checks run two different shapes
back to back through it, in both orders."""
import pytest
import torch

from paper_2606_03458_b200 import workloads as W
import kvarn_parity as P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def kv():
    from paper_2606_03458_b200 import kvarn
    return kvarn


def _case(kv, B, Hq, Hkv, n_tok, splits, seed, bits=2):
    K, V = W.kv_tokens(B, Hkv, n_tok, seed=seed, device="cuda")
    q = W.queries(B, Hq, seed=seed, device="cuda")
    p = kv.default_params(bits, splits=splits)
    cache = kv.Cache(p, B, Hkv, n_tok // 128 + 1, device="cuda", resid_dtype=K.dtype)
    kv.prefill(p, cache, K, V)
    return p, cache, q


def _close(out, ref):
    err = (out.double() - ref.double()).abs().amax(dim=-1) / ref.double().abs().amax(dim=-1).clamp_min(1e-30)
    return float(err.max())


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row(kv):
    # a: 2 clusters of 8 CTAs per (sequence, KV head) merged through the scratch (caller-chosen split), g = 4
    # b: one sequence, 2 KV heads, 40 960 tokens: the library's own plan spreads it over several clusters, g = 8
    # c: the plan of configs[1]-like shapes: one cluster, the scratch is not touched
    a = _case(kv, 2, 32, 8, 128 * 26 + 77, 16, seed=301)
    b = _case(kv, 1, 16, 2, 128 * 320 + 5, 0, seed=302)
    c = _case(kv, 2, 32, 8, 128 * 9 + 3, 0, seed=303)
    assert kv.decode_workspace_bytes(a[0], 2, 32, 8, a[1].max_chunks) > 0
    assert kv.decode_workspace_bytes(b[0], 1, 16, 2, b[1].max_chunks) > 0
    outs = {}
    # the static path FIRST (cold: its set-up must not depend on an earlier call of the other path), two calls in a row
    for name, (p, cache, q) in (("a", a), ("b", b)):
        outs[name] = kv.decode_attention_static(p, cache, q)
    torch.cuda.synchronize()
    refs = {name: kv.decode_attention(p, cache, q) for name, (p, cache, q) in (("a", a), ("b", b), ("c", c))}
    for name in ("a", "b"):
        assert _close(outs[name], refs[name]) <= P.ATTN_RTOL, name
        assert torch.equal(outs[name], refs[name]), name        # same kernel, same plan: the same bits
    # again in the other order (each call finds the other shape's partials in the array), and the untouched route
    for name, (p, cache, q) in (("b", b), ("a", a), ("c", c), ("a", a)):
        out = kv.decode_attention_static(p, cache, q)
        assert _close(out, refs[name]) <= P.ATTN_RTOL, name
        assert torch.equal(out, refs[name]), name
    # the caller's ticket array is not used by the static path
    assert int(a[1].decode_ticket.abs().sum()) == 0 and int(b[1].decode_ticket.abs().sum()) == 0


def test_static_scratch_allocates_nothing_and_rejects_oversized_plans(kv):
    p, cache, q = _case(kv, 2, 32, 8, 128 * 26 + 77, 16, seed=304)
    out = torch.empty((2, 32, 128), dtype=torch.float32, device="cuda")
    kv.decode_attention_static(p, cache, q, out=out)              # warm: module loaded, attributes set
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(4):
        kv.decode_attention_static(p, cache, q, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < (1 << 20), (free0, free1)              # no device allocation behind the call
    # 64 query heads x 2 sequences x 9 clusters x 1040 B = 1.2 MB of partials > 1 MiB - 4 KiB: refused, nothing launched
    pb, cb, qb = _case(kv, 2, 64, 8, 128 * 26 + 77, 27, seed=305)
    with pytest.raises(kv.KvarnError, match="KVARN_WORKSPACE_TOO_SMALL"):
        kv.decode_attention_static(pb, cb, qb)
    assert kv.decode_attention(pb, cb, qb).isfinite().all()        # the workspace path still serves that plan


def test_static_scratch_under_cuda_graph_capture(kv):
    """The use the entry point exists for: after one warm call, the call is captured into a CUDA graph (the counter
    clear becomes a memset node, the kernel a kernel node) and the replays reproduce the workspace path's bits."""
    p, cache, q = _case(kv, 2, 32, 8, 128 * 26 + 77, 16, seed=306)
    ref = kv.decode_attention(p, cache, q)
    out = torch.empty_like(ref)
    kv.decode_attention_static(p, cache, q, out=out)              # one-time set-up outside the capture
    torch.cuda.synchronize()
    out.zero_()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            kv.decode_attention_static(p, cache, q, out=out, stream=side)
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(2):
        out.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
