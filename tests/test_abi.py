"""CPU-only checks of the C-ABI library: it loads, exports every symbol the
header declares, validates arguments without touching a GPU, and its host-side
record pack/unpack hooks agree with the oracle's storage formats."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import kvarn_oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def kv():
    from paper_2606_03458_b200 import build
    build.build()
    from paper_2606_03458_b200 import kvarn
    return kvarn


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "kvarn.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kvarn_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported(kv):
    names = _declared_symbols()
    assert len(names) >= 12
    for n in names:
        assert hasattr(kv.lib, n), f"{n} declared in include/kvarn.h but not exported"
        assert n in kv.EXPORTS, f"{n} has no ctypes signature in the binding"


def test_no_torch_types_in_abi():
    src = open(os.path.join(ROOT, "include", "kvarn.h")).read()
    assert "torch" not in src.lower() and "at::" not in src and "#include <cuda" not in src


def test_layout_and_bit_accounting(kv):
    # 2 + (8 + 8 + 16)/128 = 2.25 bit/element; 9216 B per (chunk, KV head) for K+V
    p = kv.default_params(2)
    info = kv.layout(p)
    assert info.record_bytes == 4608 and info.codes_bytes == 4096
    assert (info.s1_off, info.s2_off, info.z_off) == (4096, 4224, 4352)
    assert 2 * info.record_bytes == 9216 and info.record_bytes * 8 / (128 * 128) == 2.25
    p4 = kv.default_params(4)
    assert kv.layout(p4).record_bytes == 8704
    assert kv.layout(p4).record_bytes * 8 / (128 * 128) == 4.25


def test_default_params_are_the_papers(kv):
    p = kv.default_params(2)
    assert (p.head_dim, p.chunk, p.bits, p.iters) == (128, 128, 2, 8)
    assert (p.log_lo, p.log_hi) == (pytest.approx(-0.3), pytest.approx(10.0))
    assert p.var_min == pytest.approx(O.VARN_C_MIN) and p.var_max == pytest.approx(O.VARN_C_MAX)
    assert p.rotate_k == 1 and p.rotate_v == 1


def test_status_strings_and_argument_validation_without_gpu(kv):
    assert kv.lib.kvarn_status_string(0) == b"KVARN_OK"
    assert kv.lib.kvarn_status_string(-2) == b"KVARN_UNSUPPORTED"
    assert kv.lib.kvarn_version() >= 1
    p = kv.default_params(3)
    info = kv.LayoutInfo()
    assert kv.lib.kvarn_layout(C.byref(p), C.byref(info)) == -2
    p = kv.default_params(2)
    # null tiles
    assert kv.lib.kvarn_quantize_chunk(C.byref(p), None, None, 1, 16384, 128, None, None, 4608, None, None) == -1
    # misaligned pointer (never dereferenced: validation happens first)
    st = kv.lib.kvarn_quantize_chunk(C.byref(p), C.c_void_p(0x1004), C.c_void_p(0x1000), 1, 16384, 128,
                                     C.c_void_p(0x2000), C.c_void_p(0x3000), 4608, None, None)
    assert st == -3
    p.head_dim = 64
    assert kv.lib.kvarn_quantize_chunk(C.byref(p), C.c_void_p(0x1000), C.c_void_p(0x1000), 1, 16384, 128,
                                       C.c_void_p(0x2000), C.c_void_p(0x3000), 4608, None, None) == -2
    p = kv.default_params(2)
    cache = kv.CacheDesc(0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 0x6000, 0x6800, 2, 8, 4, 0)
    # Hq not a multiple of Hkv, g > 8, workspace too small
    assert kv.lib.kvarn_decode_attention(C.byref(p), C.byref(cache), C.c_void_p(0x7000), 12, 0.1,
                                         C.c_void_p(0x8000), C.c_void_p(0x9000), 1 << 30, None) == -1
    assert kv.lib.kvarn_decode_attention(C.byref(p), C.byref(cache), C.c_void_p(0x7000), 128, 0.1,
                                         C.c_void_p(0x8000), C.c_void_p(0x9000), 1 << 30, None) == -2
    assert kv.lib.kvarn_decode_attention(C.byref(p), C.byref(cache), C.c_void_p(0x7000), 32, 0.1,
                                         C.c_void_p(0x8000), C.c_void_p(0x9000), 16, None) == -4
    need = kv.decode_workspace_bytes(p, 2, 32, 8, 4)
    assert need > 0 and need % 16 == 0


def test_argument_validation_of_the_later_entry_points_without_gpu(kv):
    """Every check below fails before any pointer is dereferenced or any kernel is launched."""
    L = kv.lib
    p = kv.default_params(2)
    cache = kv.CacheDesc(0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 0x6000, 0x6800, 2, 8, 4, 0)
    ptr = C.c_void_p
    # kvarn_block_attention: n_q < 1, g = 3 (not a power of two), n_q > 128, null block, misaligned q
    blk = lambda q, kb, vb, n_q, Hq: L.kvarn_block_attention(C.byref(p), C.byref(cache), q, kb, vb, n_q, Hq, 0.1, ptr(0x9000), None)
    assert blk(ptr(0x7000), ptr(0x7100), ptr(0x7200), 0, 32) == -1
    assert blk(ptr(0x7000), ptr(0x7100), ptr(0x7200), 4, 24) == -2
    assert blk(ptr(0x7000), ptr(0x7100), ptr(0x7200), 129, 32) == -2
    assert blk(ptr(0x7000), None, ptr(0x7200), 4, 32) == -1
    assert blk(ptr(0x7004), ptr(0x7100), ptr(0x7200), 4, 32) == -3
    # kvarn_append_block: n_new out of range
    assert L.kvarn_append_block(C.byref(p), C.byref(cache), ptr(0x7000), ptr(0x7100), 0, None) == -1
    assert L.kvarn_append_block(C.byref(p), C.byref(cache), ptr(0x7000), ptr(0x7100), 129, None) == -2
    # host-checkable capacity bound: capacity = n_sink + max_chunks * 128 + 127 = 639 tokens here
    full = kv.CacheDesc(0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 0x6000, 0x6800, 2, 8, 4, 0, None, None, 639, None)
    assert L.kvarn_append(C.byref(p), C.byref(full), ptr(0x7000), ptr(0x7100), None) == -5
    full.max_len_hint = 600
    assert L.kvarn_append_block(C.byref(p), C.byref(full), ptr(0x7000), ptr(0x7100), 40, None) == -5
    assert L.kvarn_status_string(-5) == b"KVARN_CAPACITY"
    # aux_round must be 0 or 1
    bad = kv.default_params(2, aux_round=2)
    assert L.kvarn_append_block(C.byref(bad), C.byref(cache), ptr(0x7000), ptr(0x7100), 1, None) == -1
    # kvarn_merge_partials
    assert L.kvarn_merge_partials(ptr(0x7000), 0, 4, ptr(0x8000), kv.F32, None) == -1
    assert L.kvarn_merge_partials(ptr(0x7000), 2, 4, ptr(0x8000), 7, None) == -2
    assert L.kvarn_merge_partials(ptr(0x7004), 2, 4, ptr(0x8000), kv.F32, None) == -3
    assert L.kvarn_merge_partials(ptr(0x7000), 2, 0, ptr(0x8000), kv.F32, None) == 0
    # rotations: cos without sin, bad dtype, rows not a multiple of 128, empty inputs are no-ops
    assert L.kvarn_rope_hadamard(ptr(0x7000), ptr(0x7100), None, ptr(0x8000), 4, 2, kv.F32, 1, None) == -1
    assert L.kvarn_rope_hadamard(ptr(0x7000), None, None, ptr(0x8000), 4, 2, 5, 1, None) == -2
    assert L.kvarn_rope_hadamard(None, None, None, None, 0, 2, kv.F32, 1, None) == 0
    assert L.kvarn_hadamard_row_groups(ptr(0x7000), ptr(0x8000), 100, 8, kv.F32, None) == -1
    assert L.kvarn_hadamard_row_groups(ptr(0x7000), ptr(0x8000), 0, 8, kv.F32, None) == 0
    assert L.kvarn_version() >= 3


@pytest.mark.parametrize("bits", [2, 4])
@pytest.mark.parametrize("kind", [0, 1])
def test_pack_unpack_round_trip_and_formats(kv, bits, kind):
    p = kv.default_params(bits)
    rng = np.random.default_rng(bits * 2 + kind)
    codes = rng.integers(0, 1 << bits, size=(128, 128)).astype(np.uint8)
    s1 = np.exp(rng.uniform(-5, 6, size=128)).astype(np.float32)
    s2 = np.exp(rng.uniform(-1, 5, size=128)).astype(np.float32)
    z = (rng.standard_normal(128) * 3).astype(np.float32)
    rec = kv.pack_record(p, kind, codes, s1, s2, z)
    assert rec.size == kv.record_bytes(p)
    c2, a1, a2, zz = kv.unpack_record(p, kind, rec)
    assert np.array_equal(c2, codes)
    # stored values are the oracle's FP8-E4M3 / FP16 roundings (reading R9)
    assert np.array_equal(a1.astype(np.float64), O.round_fp8_e4m3(s1.astype(np.float64)))
    assert np.array_equal(a2.astype(np.float64), O.round_fp8_e4m3(s2.astype(np.float64)))
    assert np.array_equal(zz.astype(np.float64), O.round_fp16(z.astype(np.float64)))
    info = kv.layout(p)
    stored = rec[info.s1_off:info.s1_off + 128]
    e = np.arange(128)
    if kind == 0:
        # K records keep s1 (and z), per channel, in the order of the B-operand builder (include/kvarn.h)
        stored = stored[_kaux_of_elem(bits, e)]
    else:
        # V records keep s1 (and z), per token, at the MMA row slot of the token
        stored = stored[_slot_of_token(bits, e)]
    assert np.array_equal(stored, O.fp8_e4m3_bits(O.round_fp8_e4m3(s1.astype(np.float64))))
    # saturation
    rec = kv.pack_record(p, kind, codes, np.full(128, 1e6, np.float32), s2, z)
    assert np.all(kv.unpack_record(p, kind, rec)[1] == 448.0)


def _kstep_kpos(bits, e):
    # include/kvarn.h "record layout": k-step and position of row element e in the contraction
    if bits == 2:
        return e & 3, 16 * (e >> 6) + 4 * ((e >> 4) & 3) + ((e >> 2) & 3)
    return 2 * (e >> 6) + (e & 1), 16 * ((e >> 5) & 1) + 4 * ((e >> 3) & 3) + ((e >> 1) & 3)


def _kaux_of_elem(bits, e):
    ks, kp = _kstep_kpos(bits, e)
    return 4 * (8 * ks + (kp >> 2)) + (kp & 3)


def _slot_of_token(bits, tau):
    # row slot 32*warp + 16*mtile + 8*rho + g with warp = k-step, (half, t') = g, b = 2*mtile + rho
    ks, kp = _kstep_kpos(bits, tau)
    b, tp, half = kp & 3, (kp >> 2) & 3, kp >> 4
    return 32 * ks + 16 * (b >> 1) + 8 * (b & 1) + 4 * half + tp


def _code_off(bits, slot, byte_in_row):
    wi, bb = byte_in_row >> 2, byte_in_row & 3
    w, mt, rho, g = slot >> 5, (slot >> 4) & 1, (slot >> 3) & 1, slot & 7
    t, q = wi & 3, wi >> 2
    if bits == 2:
        return w * 1024 + mt * 512 + (4 * g + t) * 16 + rho * 8 + q * 4 + bb
    return w * 2048 + mt * 1024 + rho * 512 + (4 * g + t) * 16 + q * 4 + bb


def test_layout_maps_are_bijections():
    for bits in (2, 4):
        e = np.arange(128)
        assert sorted(_kaux_of_elem(bits, e).tolist()) == list(range(128))
        assert sorted(_slot_of_token(bits, e).tolist()) == list(range(128))
        rb = 128 * bits // 8
        offs = sorted(_code_off(bits, s, b) for s in range(128) for b in range(rb))
        assert offs == list(range(128 * rb))


def test_code_row_layout(kv):
    # include/kvarn.h: K rows are per token, V rows per channel, little-endian within a row (element e
    # at bit bits*(e % (8/bits)) of byte e*bits/8); row slot / word placement as restated above.
    p = kv.default_params(2)
    codes = np.zeros((128, 128), np.uint8)
    codes[5, 9] = 3          # token 5, channel 9
    codes[7, 100] = 2        # token 7, channel 100 -> byte 25 of its K row
    ones = np.ones(128, np.float32)
    rk = kv.pack_record(p, 0, codes, ones, ones, ones)
    rv = kv.pack_record(p, 1, codes, ones, ones, ones)
    assert rk[_code_off(2, int(_slot_of_token(2, 5)), 9 // 4)] == 3 << (2 * (9 % 4))
    assert rk[_code_off(2, int(_slot_of_token(2, 7)), 100 // 4)] == 2 << (2 * (100 % 4))
    assert rk[:4096].sum() == (3 << 2) + (2 << 0)
    assert rv[_code_off(2, 9, 5 // 4)] == 3 << (2 * (5 % 4))      # V rows: slot = channel
    assert rv[_code_off(2, 100, 7 // 4)] == 2 << (2 * (7 % 4))
    p4 = kv.default_params(4)
    r4 = kv.pack_record(p4, 0, codes, ones, ones, ones)
    assert r4[_code_off(4, int(_slot_of_token(4, 7)), 100 // 2)] == 2 << (4 * (100 % 2))
    # a random record round-trips through the canonical view at both widths
    rng = np.random.default_rng(3)
    for bits, pp in ((2, p), (4, p4)):
        c = rng.integers(0, 1 << bits, size=(128, 128)).astype(np.uint8)
        for kind in (0, 1):
            assert np.array_equal(kv.unpack_record(pp, kind, kv.pack_record(pp, kind, c, ones, ones, ones))[0], c)


def test_missing_library_fails_loudly(tmp_path, monkeypatch):
    # no CPU fallback: loading the binding without the .so raises
    import importlib.util
    src = os.path.join(ROOT, "paper_2606_03458_b200", "kvarn.py")
    dst = tmp_path / "kvarn_copy.py"
    dst.write_text(open(src).read())
    spec = importlib.util.spec_from_file_location("kvarn_copy", dst)
    mod = importlib.util.module_from_spec(spec)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        spec.loader.exec_module(mod)


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_03458_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("oracle-side", "").replace("the oracle", "").replace("oracle and", "") \
                    or "import oracle" not in txt and "from oracle" not in txt, f
                assert "from oracle" not in txt and "import oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "kvarn_oracle.py")).read()
    assert "paper_2606_03458_b200" not in otxt.split('"""')[2]
