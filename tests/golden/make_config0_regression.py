"""Writes tests/golden/config0_oracle_regression.txt from oracle/ alone (no CUDA path involved):
a regression lock on the oracle's own output for BASELINE.json configs[0], so that an accidental change
to the oracle's arithmetic shows up as a diff of a committed text file.  Not a pin (the oracle checks itself).

    python tests/golden/make_config0_regression.py
"""
import os
import sys
import zlib

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import kvarn_oracle as O                      # noqa: E402
from paper_2606_03458_b200 import workloads as W          # noqa: E402  (seeded inputs only, no KVarN arithmetic)


def lines():
    K, V, q, _ = W.config0()
    out = []
    for bits in (2, 4):
        for name, X in (("k", K), ("v", V)):
            r = O.quantize_tile(X.astype(np.float64), name, bits=bits)
            c = np.ascontiguousarray(r.codes.astype(np.uint8))
            out.append(f"{name}{bits}.k_best = {r.k_best}")
            out.append(f"{name}{bits}.codes_crc32 = {zlib.crc32(c.tobytes())}")
            out.append(f"{name}{bits}.codes_hist = {' '.join(str(int(x)) for x in np.bincount(c.ravel(), minlength=1 << bits))}")
            out.append(f"{name}{bits}.s1_sum = {float(np.sum(r.s1)):.10g}")
            out.append(f"{name}{bits}.s2_sum = {float(np.sum(r.s2)):.10g}")
            out.append(f"{name}{bits}.z_sum = {float(np.sum(r.z)):.10g}")
            out.append(f"{name}{bits}.I = {' '.join(f'{x:.8g}' for x in r.varn.I)}")
    rk, rv = O.quantize_tile(K.astype(np.float64), "k"), O.quantize_tile(V.astype(np.float64), "v")
    f = lambda a: np.asarray(a, dtype=np.float64)
    att = O.decode_attention(f(q)[None], [(rk.codes, f(rk.s1), f(rk.s2), f(rk.z))], [(rv.codes, f(rv.s1), f(rv.s2), f(rv.z))],
                             np.zeros((0, 128)), np.zeros((0, 128)))
    out.append(f"attn2.out_first8 = {' '.join(f'{x:.10g}' for x in att[0, :8])}")
    out.append(f"attn2.out_abs_sum = {float(np.abs(att).sum()):.10g}")
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_oracle_regression.txt")
    with open(path, "w") as fh:
        fh.write("# written by tests/golden/make_config0_regression.py (oracle/ only); BASELINE.json configs[0]\n")
        fh.write("\n".join(lines()) + "\n")
    print(path)
