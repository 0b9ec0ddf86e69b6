"""Derive the golden vectors G1 (KV kind) and G2 (MLA kind) of SURVEY.md §8(c) WITHOUT the
oracle and without the CUDA path: exact rational dot products (fractions.Fraction),
math.exp / math.fsum for the softmax.  Running it rewrites g1_kv.txt / g2_mla.txt; the
committed files must not change (tests/test_oracle_pins.py::test_golden_files_rederive).

All inputs are small dyadic rationals, exactly representable in bf16, so the only
rounding is in exp / the final sums (~1e-16), far below the 1e-11 pin tolerance.
"""
import math
import os
from fractions import Fraction as F

HERE = os.path.dirname(os.path.abspath(__file__))


def softmax_attend(q_rows, k_rows, v_rows, sigma):
    outs, lses, dots = [], [], []
    for q in q_rows:
        d = [sum(a * b for a, b in zip(q, k)) for k in k_rows]        # exact
        dots.append(d)
        s = [sigma * float(x) for x in d]
        m = max(s)
        p = [math.exp(x - m) for x in s]
        l = math.fsum(p)
        outs.append([math.fsum(pi * float(v[j]) for pi, v in zip(p, v_rows)) / l
                     for j in range(len(v_rows[0]))])
        lses.append(m + math.log(l))
    return dots, lses, outs


def g1():
    Hq, d, T = 2, 8, 5
    Q = [[F(((7 * h + 3 * i) % 5) - 2, 2) for i in range(d)] for h in range(Hq)]
    K = [[F(((5 * t + 11 * i) % 7) - 3, 4) for i in range(d)] for t in range(T)]
    V = [[F(((4 * t + 5 * i) % 9) - 4, 8) for i in range(d)] for t in range(T)]
    return Q, K, V, 1.0 / math.sqrt(8.0)


def g2():
    Hq, w, dv, T = 3, 6, 4, 4
    Q = [[F(((5 * h + 2 * i) % 7) - 3, 4) for i in range(w)] for h in range(Hq)]
    C = [[F(((3 * t + 5 * i) % 11) - 5, 8) for i in range(w)] for t in range(T)]
    V = [row[:dv] for row in C]
    return Q, C, V, 1.0 / math.sqrt(3.0)


def render(name, cite, Q, K, V, sigma):
    import struct
    sigma32 = struct.unpack("f", struct.pack("f", sigma))[0]   # the float32 both sides receive
    dots, lses, outs = softmax_attend(Q, K, V, sigma32)
    lines = ["# %s" % name, "# source: %s" % cite,
             "# derived by tests/golden/make_golden.py (Fraction dot products, math.exp/fsum)"]
    for h, d in enumerate(dots):
        lines.append("dots %d %s" % (h, " ".join(str(x) for x in d)))
    lines.append("# sigma = float32(%r) widened to double: what both the oracle and the GPU receive" % sigma)
    lines.append("lse " + " ".join("%.15f" % x for x in lses))
    for h, o in enumerate(outs):
        lines.append("out %d %s" % (h, " ".join("%.15f" % x for x in o)))
    # the same with the unrounded double sigma: these are the digits SURVEY.md §8(c) prints
    _, lses64, outs64 = softmax_attend(Q, K, V, sigma)
    lines.append("# sigma as an unrounded double (the 12 digits printed in SURVEY.md §8(c))")
    lines.append("lse_sigma64 " + " ".join("%.12f" % x for x in lses64))
    for h, o in enumerate(outs64):
        lines.append("out_sigma64 %d %s" % (h, " ".join("%.12f" % x for x in o)))
    return "\n".join(lines) + "\n"


def main(write=True):
    texts = {
        "g1_kv.txt": render("G1: KV kind, Hq=2 Hkv=1 d=8 T=5 P=2 sigma=1/sqrt(8)",
                            "SURVEY.md §8(c) golden vector G1 (no value on this path is printed "
                            "by PAPER.md; see DESIGN.md §3)", *g1()),
        "g2_mla.txt": render("G2: MLA kind, Hq=3 width=6 d_v=4 T=4 P=2 sigma=1/sqrt(3)",
                             "SURVEY.md §8(c) golden vector G2", *g2()),
    }
    if write:
        for fn, t in texts.items():
            with open(os.path.join(HERE, fn), "w") as f:
                f.write(t)
    return texts


if __name__ == "__main__":
    main()
