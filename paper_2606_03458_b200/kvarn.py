"""Thin ctypes binding of libkvarn.so (include/kvarn.h) -- argument marshalling only.

Every step of the KVarN hot path runs inside the CUDA library; this module
turns torch tensors into device pointers, fills the POD structs and checks the
returned status.  There is no CPU fallback: importing this module without a
built library raises, and every call raises on a non-zero status.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkvarn.so")

HEAD_DIM = 128
CHUNK = 128
MAX_ITERS = 16
BF16, F32 = 0, 1
KIND_K, KIND_V = 0, 1


class KvarnError(RuntimeError):
    pass


class Params(C.Structure):
    _fields_ = [("head_dim", C.c_int32), ("chunk", C.c_int32), ("bits", C.c_int32),
                ("iters", C.c_int32), ("var_min", C.c_float), ("var_max", C.c_float),
                ("log_lo", C.c_float), ("log_hi", C.c_float), ("rotate_k", C.c_int32),
                ("rotate_v", C.c_int32), ("in_dtype", C.c_int32), ("out_dtype", C.c_int32),
                ("splits", C.c_int32), ("aux_round", C.c_int32), ("decode_digits", C.c_int32)]


class LayoutInfo(C.Structure):
    _fields_ = [("record_bytes", C.c_size_t), ("codes_off", C.c_size_t),
                ("codes_bytes", C.c_size_t), ("s1_off", C.c_size_t), ("s2_off", C.c_size_t),
                ("z_off", C.c_size_t)]


class CacheDesc(C.Structure):
    _fields_ = [("k_records", C.c_void_p), ("v_records", C.c_void_p), ("k_resid", C.c_void_p),
                ("v_resid", C.c_void_p), ("seq_lens", C.c_void_p), ("ticket", C.c_void_p),
                ("decode_ticket", C.c_void_p), ("B", C.c_int32), ("Hkv", C.c_int32), ("max_chunks", C.c_int32),
                ("n_sink", C.c_int32), ("k_sink", C.c_void_p), ("v_sink", C.c_void_p),
                ("max_len_hint", C.c_int32), ("overflow", C.c_void_p)]


class DebugDesc(C.Structure):
    _fields_ = [("k_best", C.c_void_p), ("imb", C.c_void_p), ("aux_f32", C.c_void_p)]


EXPORTS = {
    "kvarn_default_params": (None, [C.POINTER(Params), C.c_int32]),
    "kvarn_status_string": (C.c_char_p, [C.c_int]),
    "kvarn_version": (C.c_int, []),
    "kvarn_layout": (C.c_int, [C.POINTER(Params), C.POINTER(LayoutInfo)]),
    "kvarn_decode_workspace_bytes": (C.c_size_t, [C.POINTER(Params), C.c_int32, C.c_int32, C.c_int32, C.c_int32]),
    "kvarn_decode_attention_static": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_int32, C.c_float,
                                                C.c_void_p, C.c_void_p]),
    "kvarn_quantize_chunk": (C.c_int, [C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_int64, C.c_int64,
                                       C.c_int64, C.c_void_p, C.c_void_p, C.c_int64,
                                       C.POINTER(DebugDesc), C.c_void_p]),
    "kvarn_prefill": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_void_p,
                                C.c_int32, C.c_void_p]),
    "kvarn_append": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_void_p, C.c_void_p]),
    "kvarn_append_block": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_void_p, C.c_int32,
                                     C.c_void_p]),
    "kvarn_decode_attention": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_int32,
                                         C.c_float, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]),
    "kvarn_block_attention": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_int32, C.c_int32, C.c_float, C.c_void_p, C.c_void_p]),
    "kvarn_block_dense_workspace_bytes": (C.c_size_t, [C.POINTER(Params), C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32]),
    "kvarn_block_attention_dense": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_void_p,
                                              C.c_void_p, C.c_int32, C.c_int32, C.c_float, C.c_void_p, C.c_void_p,
                                              C.c_size_t, C.c_void_p]),
    "kvarn_rope_hadamard": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32,
                                      C.c_int32, C.c_int32, C.c_void_p]),
    "kvarn_hadamard_rows": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_void_p]),
    "kvarn_hadamard_row_groups": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int32, C.c_void_p]),
    "kvarn_decode_attention_partial": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_int32,
                                                 C.c_float, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]),
    "kvarn_merge_partials": (C.c_int, [C.c_void_p, C.c_int32, C.c_int64, C.c_void_p, C.c_int32, C.c_void_p]),
    "kvarn_quantize_chunk_host": (C.c_int, [C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_int64] +
                                  [C.c_void_p] * 7),
    "kvarn_decode_attention_host": (C.c_int, [C.POINTER(Params), C.POINTER(CacheDesc), C.c_void_p, C.c_int32,
                                              C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                              C.c_size_t, C.c_void_p]),
    "kvarn_unpack_record_host": (C.c_int, [C.POINTER(Params), C.c_int32, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.c_void_p, C.c_void_p]),
    "kvarn_pack_record_host": (C.c_int, [C.POINTER(Params), C.c_int32, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p]),
}


def _load():
    if not os.path.exists(LIB_PATH):
        raise KvarnError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2606_03458_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    for name, (res, args) in EXPORTS.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    return lib


lib = _load()


def _check(status: int, what: str):
    if status != 0:
        raise KvarnError(f"{what}: {lib.kvarn_status_string(status).decode()} ({status})")


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.bfloat16:
        return BF16
    if t.dtype == torch.float32:
        return F32
    raise KvarnError(f"unsupported dtype {t.dtype}")


def default_params(bits: int = 2, **overrides) -> Params:
    p = Params()
    lib.kvarn_default_params(C.byref(p), bits)
    for k, v in overrides.items():
        setattr(p, k, v)
    return p


def layout(p: Params) -> LayoutInfo:
    info = LayoutInfo()
    _check(lib.kvarn_layout(C.byref(p), C.byref(info)), "kvarn_layout")
    return info


def record_bytes(p: Params) -> int:
    return int(layout(p).record_bytes)


class QuantDebug:
    def __init__(self, n_tiles: int, device):
        self.k_best = torch.zeros((2, n_tiles), dtype=torch.int32, device=device)
        self.imb = torch.zeros((2, n_tiles, MAX_ITERS + 1), dtype=torch.float32, device=device)
        self.aux = torch.zeros((2, n_tiles, 3, 128), dtype=torch.float32, device=device)
        self.desc = DebugDesc(self.k_best.data_ptr(), self.imb.data_ptr(), self.aux.data_ptr())


def quantize_chunk(p: Params, k: torch.Tensor | None, v: torch.Tensor | None, k_rec=None, v_rec=None,
                   debug: bool = False, stream=None):
    """k, v: [n_tiles, 128, 128] (token-major tiles, contiguous).  Returns
    (k_rec, v_rec[, QuantDebug]) with records as uint8 [n_tiles, record_bytes]."""
    ref = k if k is not None else v
    n_tiles = ref.shape[0]
    for t in (k, v):
        if t is not None:
            assert t.is_cuda and t.is_contiguous() and tuple(t.shape[1:]) == (CHUNK, HEAD_DIM)
    p.in_dtype = _dtype_code(ref)
    rb = record_bytes(p)
    if k is not None and k_rec is None:
        k_rec = torch.empty((n_tiles, rb), dtype=torch.uint8, device=ref.device)
    if v is not None and v_rec is None:
        v_rec = torch.empty((n_tiles, rb), dtype=torch.uint8, device=ref.device)
    dbg = QuantDebug(n_tiles, ref.device) if debug else None
    st = lib.kvarn_quantize_chunk(C.byref(p), _ptr(k), _ptr(v), n_tiles, CHUNK * HEAD_DIM, HEAD_DIM,
                                  _ptr(k_rec), _ptr(v_rec), rb,
                                  C.byref(dbg.desc) if dbg else None, _stream(stream))
    _check(st, "kvarn_quantize_chunk")
    return (k_rec, v_rec, dbg) if debug else (k_rec, v_rec)


class Cache:
    """Device buffers of one layer's KVarN cache + the POD descriptor."""

    def __init__(self, p: Params, B: int, Hkv: int, max_chunks: int, device="cuda",
                 resid_dtype=torch.bfloat16, n_sink: int = 0):
        """n_sink = S of the paper's three-region layout: the first S tokens of every sequence
        stay raw (0 = no sink region; the paper uses 128, and 32 for IFEval)."""
        rb = record_bytes(p)
        self.B, self.Hkv, self.max_chunks, self.rb, self.n_sink = B, Hkv, max_chunks, rb, n_sink
        self.k_sink = torch.zeros((B, Hkv, max(n_sink, 1), HEAD_DIM), dtype=resid_dtype, device=device)
        self.v_sink = torch.zeros_like(self.k_sink)
        self.k_records = torch.zeros((B, Hkv, max(max_chunks, 1), rb), dtype=torch.uint8, device=device)
        self.v_records = torch.zeros_like(self.k_records)
        self.k_resid = torch.zeros((B, Hkv, CHUNK, HEAD_DIM), dtype=resid_dtype, device=device)
        self.v_resid = torch.zeros_like(self.k_resid)
        self.seq_lens = torch.zeros((B,), dtype=torch.int32, device=device)
        self.ticket = torch.zeros((B,), dtype=torch.int32, device=device)
        self.decode_ticket = torch.zeros((B * Hkv,), dtype=torch.int32, device=device)
        self.overflow = torch.zeros((1,), dtype=torch.int32, device=device)
        self.desc = CacheDesc(self.k_records.data_ptr(), self.v_records.data_ptr(),
                              self.k_resid.data_ptr(), self.v_resid.data_ptr(),
                              self.seq_lens.data_ptr(), self.ticket.data_ptr(),
                              self.decode_ticket.data_ptr(), B, Hkv, max_chunks, n_sink,
                              self.k_sink.data_ptr(), self.v_sink.data_ptr(), 0, self.overflow.data_ptr())

    def slice(self, b0: int, b1: int) -> "Cache":
        """A cache over sequences b0..b1-1 that shares this cache's buffers (views, no copy):
        lets a large cache be filled or read a few sequences at a time."""
        assert 0 <= b0 < b1 <= self.B, (b0, b1, self.B)
        c = Cache.__new__(Cache)
        c.B, c.Hkv, c.max_chunks, c.rb, c.n_sink = b1 - b0, self.Hkv, self.max_chunks, self.rb, self.n_sink
        c.k_sink, c.v_sink = self.k_sink[b0:b1], self.v_sink[b0:b1]
        c.k_records, c.v_records = self.k_records[b0:b1], self.v_records[b0:b1]
        c.k_resid, c.v_resid = self.k_resid[b0:b1], self.v_resid[b0:b1]
        c.seq_lens, c.ticket = self.seq_lens[b0:b1], self.ticket[b0:b1]
        c.decode_ticket = self.decode_ticket[b0 * self.Hkv:b1 * self.Hkv]
        c.overflow = self.overflow
        c.desc = CacheDesc(c.k_records.data_ptr(), c.v_records.data_ptr(), c.k_resid.data_ptr(),
                           c.v_resid.data_ptr(), c.seq_lens.data_ptr(), c.ticket.data_ptr(),
                           c.decode_ticket.data_ptr(), c.B, c.Hkv, c.max_chunks, c.n_sink,
                           c.k_sink.data_ptr(), c.v_sink.data_ptr(), 0, c.overflow.data_ptr())
        return c

    def nbytes_read_by_decode(self, ctx: int) -> int:
        """Algorithmic bytes one decode step reads for context length ctx."""
        ns = min(ctx, self.n_sink)
        n_chunks, r = (ctx - ns) // CHUNK, (ctx - ns) % CHUNK
        es = self.k_resid.element_size()
        return self.B * self.Hkv * (n_chunks * 2 * self.rb + (r + ns) * 2 * HEAD_DIM * es)


def prefill(p: Params, cache: Cache, k: torch.Tensor, v: torch.Tensor, stream=None):
    """k, v: [B, Hkv, n_tok, 128]."""
    assert k.is_cuda and k.is_contiguous() and v.is_contiguous() and k.shape == v.shape
    assert tuple(k.shape[:2]) == (cache.B, cache.Hkv) and k.shape[3] == HEAD_DIM
    p.in_dtype = _dtype_code(k)
    assert cache.k_resid.dtype == k.dtype
    _check(lib.kvarn_prefill(C.byref(p), C.byref(cache.desc), _ptr(k), _ptr(v), k.shape[2],
                             _stream(stream)), "kvarn_prefill")


def append(p: Params, cache: Cache, k_new: torch.Tensor, v_new: torch.Tensor, stream=None, max_len_hint: int = 0):
    """k_new, v_new: [B, Hkv, 128] -- one new token per sequence.  max_len_hint > 0: the caller's upper bound on
    the sequence lengths before the call (KVARN_CAPACITY is raised when the token provably cannot fit)."""
    assert k_new.is_cuda and k_new.is_contiguous() and v_new.is_contiguous()
    assert tuple(k_new.shape) == (cache.B, cache.Hkv, HEAD_DIM) and k_new.shape == v_new.shape
    p.in_dtype = _dtype_code(k_new)
    assert cache.k_resid.dtype == k_new.dtype
    cache.desc.max_len_hint = int(max_len_hint)
    _check(lib.kvarn_append(C.byref(p), C.byref(cache.desc), _ptr(k_new), _ptr(v_new),
                            _stream(stream)), "kvarn_append")


def append_block(p: Params, cache: Cache, k_new: torch.Tensor, v_new: torch.Tensor, stream=None, max_len_hint: int = 0):
    """k_new, v_new: [B, Hkv, n_new, 128], 1 <= n_new <= 128 new tokens per sequence (Fig. 4)."""
    assert k_new.is_cuda and k_new.is_contiguous() and v_new.is_contiguous() and k_new.shape == v_new.shape
    assert k_new.dim() == 4 and tuple(k_new.shape[:2]) == (cache.B, cache.Hkv) and k_new.shape[3] == HEAD_DIM
    p.in_dtype = _dtype_code(k_new)
    assert cache.k_resid.dtype == k_new.dtype
    cache.desc.max_len_hint = int(max_len_hint)
    _check(lib.kvarn_append_block(C.byref(p), C.byref(cache.desc), _ptr(k_new), _ptr(v_new), k_new.shape[2],
                                  _stream(stream)), "kvarn_append_block")


def decode_workspace_bytes(p: Params, B: int, Hq: int, Hkv: int, max_chunks: int) -> int:
    return int(lib.kvarn_decode_workspace_bytes(C.byref(p), B, Hq, Hkv, max_chunks))


def decode_attention(p: Params, cache: Cache, q: torch.Tensor, sm_scale: float | None = None,
                     out: torch.Tensor | None = None, ws: torch.Tensor | None = None, stream=None):
    """q: [B, Hq, 128] -> out [B, Hq, 128] (fp32 unless p.out_dtype says bf16)."""
    assert q.is_cuda and q.is_contiguous() and q.shape[0] == cache.B and q.shape[2] == HEAD_DIM
    Hq = q.shape[1]
    p.in_dtype = _dtype_code(q)
    assert cache.k_resid.dtype == q.dtype
    if sm_scale is None:
        sm_scale = 1.0 / float(np.sqrt(HEAD_DIM))
    if out is None:
        out = torch.empty((cache.B, Hq, HEAD_DIM), device=q.device,
                          dtype=torch.float32 if p.out_dtype == F32 else torch.bfloat16)
    if ws is None:
        ws = torch.empty((max(decode_workspace_bytes(p, cache.B, Hq, cache.Hkv, cache.max_chunks), 16),),
                         dtype=torch.uint8, device=q.device)
    st = lib.kvarn_decode_attention(C.byref(p), C.byref(cache.desc), _ptr(q), Hq, sm_scale, _ptr(out),
                                    _ptr(ws), ws.numel(), _stream(stream))
    _check(st, "kvarn_decode_attention")
    return out


STATIC_SCRATCH_BYTES = 1 << 20


def decode_attention_static(p: Params, cache: Cache, q: torch.Tensor, sm_scale: float | None = None,
                            out: torch.Tensor | None = None, stream=None):
    """kvarn_decode_attention_static: decode_attention with the split-K scratch in the library's static device array
    (1 MiB per GPU; nothing is allocated by the call -- pass `out` to keep the binding allocation-free too).  Calls
    that overlap on the GPU race on that array."""
    assert q.is_cuda and q.is_contiguous() and q.shape[0] == cache.B and q.shape[2] == HEAD_DIM
    Hq = q.shape[1]
    p.in_dtype = _dtype_code(q)
    assert cache.k_resid.dtype == q.dtype
    if sm_scale is None:
        sm_scale = 1.0 / float(np.sqrt(HEAD_DIM))
    if out is None:
        out = torch.empty((cache.B, Hq, HEAD_DIM), device=q.device,
                          dtype=torch.float32 if p.out_dtype == F32 else torch.bfloat16)
    st = lib.kvarn_decode_attention_static(C.byref(p), C.byref(cache.desc), _ptr(q), Hq, sm_scale, _ptr(out), _stream(stream))
    _check(st, "kvarn_decode_attention_static")
    return out


PART_STRIDE = 132


def decode_attention_partial(p: Params, cache: Cache, q: torch.Tensor, sm_scale: float | None = None,
                             part: torch.Tensor | None = None, ws: torch.Tensor | None = None, stream=None):
    """q: [B, Hq, 128] -> part [B, Hq, 132] fp32 = {m, l, 0, 0, o[128]}: this cache's un-normalised share of the
    attention (context-parallel building block)."""
    assert q.is_cuda and q.is_contiguous() and q.shape[0] == cache.B and q.shape[2] == HEAD_DIM
    Hq = q.shape[1]
    p.in_dtype = _dtype_code(q)
    assert cache.k_resid.dtype == q.dtype
    if sm_scale is None:
        sm_scale = 1.0 / float(np.sqrt(HEAD_DIM))
    if part is None:
        part = torch.empty((cache.B, Hq, PART_STRIDE), device=q.device, dtype=torch.float32)
    if ws is None:
        ws = torch.empty((max(decode_workspace_bytes(p, cache.B, Hq, cache.Hkv, cache.max_chunks), 16),),
                         dtype=torch.uint8, device=q.device)
    st = lib.kvarn_decode_attention_partial(C.byref(p), C.byref(cache.desc), _ptr(q), Hq, sm_scale, _ptr(part),
                                            _ptr(ws), ws.numel(), _stream(stream))
    _check(st, "kvarn_decode_attention_partial")
    return part


def merge_partials(parts: torch.Tensor, out_dtype=torch.float32, out: torch.Tensor | None = None, stream=None):
    """parts: [R, B, Hq, 132] fp32 (the ranks' partials, all-gathered) -> out [B, Hq, 128]."""
    assert parts.is_cuda and parts.is_contiguous() and parts.dtype == torch.float32 and parts.shape[-1] == PART_STRIDE
    R, B, Hq = parts.shape[:3]
    if out is None:
        out = torch.empty((B, Hq, HEAD_DIM), device=parts.device, dtype=out_dtype)
    _check(lib.kvarn_merge_partials(_ptr(parts), R, B * Hq, _ptr(out), F32 if out.dtype == torch.float32 else BF16,
                                    _stream(stream)), "kvarn_merge_partials")
    return out


def context_parallel_decode(p: Params, cache: Cache, q: torch.Tensor, group=None, sm_scale: float | None = None):
    """One decode step with every sequence's tokens split across the ranks of `group` (each rank's `cache` holds its
    share): local partial -> all_gather_into_tensor (NCCL over NVLink) -> LSE merge.  Every rank gets the output."""
    import torch.distributed as dist
    part = decode_attention_partial(p, cache, q, sm_scale=sm_scale)
    world = dist.get_world_size(group)
    parts = torch.empty((world,) + tuple(part.shape), device=part.device, dtype=torch.float32)
    dist.all_gather_into_tensor(parts, part, group=group)       # 528 B per (b, q head) and rank
    return merge_partials(parts, out_dtype=torch.float32 if p.out_dtype == F32 else torch.bfloat16)


def block_attention(p: Params, cache: Cache, q: torch.Tensor, k_blk: torch.Tensor, v_blk: torch.Tensor,
                    sm_scale: float | None = None, out: torch.Tensor | None = None, stream=None,
                    dense: bool = False, ws: torch.Tensor | None = None):
    """q: [B, n_q, Hq, 128]; k_blk, v_blk: [B, Hkv, n_q, 128] (the block's own raw tokens, not yet in
    the cache) -> out [B, n_q, Hq, 128]: causal attention over [cache ; block] (Fig. 4)."""
    assert q.is_cuda and q.is_contiguous() and q.shape[0] == cache.B and q.shape[3] == HEAD_DIM
    n_q, Hq = q.shape[1], q.shape[2]
    assert k_blk.is_contiguous() and v_blk.is_contiguous() and k_blk.shape == v_blk.shape
    assert tuple(k_blk.shape) == (cache.B, cache.Hkv, n_q, HEAD_DIM) and k_blk.dtype == q.dtype
    p.in_dtype = _dtype_code(q)
    assert cache.k_resid.dtype == q.dtype
    if sm_scale is None:
        sm_scale = 1.0 / float(np.sqrt(HEAD_DIM))
    if out is None:
        out = torch.empty((cache.B, n_q, Hq, HEAD_DIM), device=q.device,
                          dtype=torch.float32 if p.out_dtype == F32 else torch.bfloat16)
    if dense:   # the tcgen05 form (kvarn_block_attention_dense): for blocks with many (token, head) rows per KV head
        if ws is None:
            need = int(lib.kvarn_block_dense_workspace_bytes(C.byref(p), cache.B, Hq, cache.Hkv, n_q, cache.max_chunks))
            ws = torch.empty((max(need, 16),), dtype=torch.uint8, device=q.device)
        st = lib.kvarn_block_attention_dense(C.byref(p), C.byref(cache.desc), _ptr(q), _ptr(k_blk), _ptr(v_blk), n_q, Hq,
                                             sm_scale, _ptr(out), _ptr(ws), ws.numel(), _stream(stream))
        _check(st, "kvarn_block_attention_dense")
        return out
    st = lib.kvarn_block_attention(C.byref(p), C.byref(cache.desc), _ptr(q), _ptr(k_blk), _ptr(v_blk), n_q, Hq,
                                   sm_scale, _ptr(out), _stream(stream))
    _check(st, "kvarn_block_attention")
    return out


def rope_hadamard(x: torch.Tensor, cos: torch.Tensor | None = None, sin: torch.Tensor | None = None,
                  rotate: bool = True, out: torch.Tensor | None = None, stream=None):
    """x: [n_tok, n_heads, 128]; cos, sin: fp32 [n_tok, 64] or None -> RoPE(x) H / sqrt(128) (App. A)."""
    assert x.is_cuda and x.is_contiguous() and x.dim() == 3 and x.shape[2] == HEAD_DIM
    if cos is not None:
        assert cos.dtype == torch.float32 and sin.dtype == torch.float32 and cos.is_contiguous() and sin.is_contiguous()
        assert tuple(cos.shape) == (x.shape[0], HEAD_DIM // 2) and cos.shape == sin.shape
    out = torch.empty_like(x) if out is None else out
    _check(lib.kvarn_rope_hadamard(_ptr(x), _ptr(cos), _ptr(sin), _ptr(out), x.shape[0], x.shape[1], _dtype_code(x),
                                   int(rotate), _stream(stream)), "kvarn_rope_hadamard")
    return out


def hadamard_rows(x: torch.Tensor, out: torch.Tensor | None = None, stream=None):
    """Rotate every 128-element group of a contiguous tensor whose last dimension is a multiple of 128."""
    assert x.is_cuda and x.is_contiguous() and x.shape[-1] % HEAD_DIM == 0
    out = torch.empty_like(x) if out is None else out
    _check(lib.kvarn_hadamard_rows(_ptr(x), _ptr(out), x.numel() // HEAD_DIM, _dtype_code(x), _stream(stream)),
           "kvarn_hadamard_rows")
    return out


def hadamard_row_groups(w: torch.Tensor, out: torch.Tensor | None = None, stream=None):
    """w: [n_rows, n_cols], n_rows % 128 == 0 -> blockdiag(H / sqrt(128)) w (the absorbed transform of W_O)."""
    assert w.is_cuda and w.is_contiguous() and w.dim() == 2
    out = torch.empty_like(w) if out is None else out
    _check(lib.kvarn_hadamard_row_groups(_ptr(w), _ptr(out), w.shape[0], w.shape[1], _dtype_code(w), _stream(stream)),
           "kvarn_hadamard_row_groups")
    return out


def quantize_chunk_host(p: Params, k_host, v_host, dev_in_k, dev_in_v, dev_rec_k, dev_rec_v,
                        k_rec_host=None, v_rec_host=None, stream=None):
    """HOST k, v [n_tiles,128,128] -> device records (+ optional HOST copies)."""
    n_tiles = k_host.shape[0]
    p.in_dtype = _dtype_code(k_host)
    st = lib.kvarn_quantize_chunk_host(C.byref(p), _ptr(k_host), _ptr(v_host), n_tiles, _ptr(dev_in_k),
                                       _ptr(dev_in_v), _ptr(dev_rec_k), _ptr(dev_rec_v),
                                       _ptr(k_rec_host), _ptr(v_rec_host), _stream(stream))
    _check(st, "kvarn_quantize_chunk_host")


def decode_attention_host(p: Params, cache: Cache, q_host, out_host, dev_q, dev_out, ws,
                          sm_scale: float | None = None, stream=None):
    Hq = q_host.shape[1]
    p.in_dtype = _dtype_code(q_host)
    if sm_scale is None:
        sm_scale = 1.0 / float(np.sqrt(HEAD_DIM))
    st = lib.kvarn_decode_attention_host(C.byref(p), C.byref(cache.desc), _ptr(q_host), Hq, sm_scale,
                                         _ptr(out_host), _ptr(dev_q), _ptr(dev_out), _ptr(ws), ws.numel(),
                                         _stream(stream))
    _check(st, "kvarn_decode_attention_host")


def unpack_record(p: Params, kind: int, record: np.ndarray):
    """Host test hook: record bytes -> (codes[t,c] u8, s1, s2, z as fp32)."""
    record = np.ascontiguousarray(record, dtype=np.uint8)
    assert record.size == record_bytes(p)
    codes = np.empty((CHUNK, HEAD_DIM), dtype=np.uint8)
    s1, s2, z = (np.empty(128, dtype=np.float32) for _ in range(3))
    st = lib.kvarn_unpack_record_host(C.byref(p), kind, record.ctypes.data, codes.ctypes.data,
                                      s1.ctypes.data, s2.ctypes.data, z.ctypes.data)
    _check(st, "kvarn_unpack_record_host")
    return codes, s1, s2, z


def pack_record(p: Params, kind: int, codes: np.ndarray, s1, s2, z) -> np.ndarray:
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    s1, s2, z = (np.ascontiguousarray(a, dtype=np.float32) for a in (s1, s2, z))
    rec = np.empty(record_bytes(p), dtype=np.uint8)
    st = lib.kvarn_pack_record_host(C.byref(p), kind, codes.ctypes.data, s1.ctypes.data, s2.ctypes.data,
                                    z.ctypes.data, rec.ctypes.data)
    _check(st, "kvarn_pack_record_host")
    return rec
