"""Writes tests/golden/s2_box_integrals.txt: reference values of

    int_{t1}^{t2} int_{s1}^{s2} ds dt / sqrt(A s^2 + B s t + C t^2)

(one term of S2, eq. (21), integrated as in eq. (23)) by
mpmath tanh-sinh quadrature at 30 digits, splitting each box at the singular
point (0,0).  Uses mpmath only: nothing from oracle/ and nothing from the CUDA
path.  The paper states only that I "can be evaluated exactly in terms of
logarithms" (L187); these numbers pin the closed form the oracle uses.

Run:  python tests/golden/make_s2_box_golden.py
"""
from pathlib import Path

import mpmath as mp

mp.mp.dps = 30

# A, B, C, s1, s2, t1, t2   (A = 1 + zx^2, B = 2 zx zy, C = 1 + zy^2  =>  4AC - B^2 > 0)
CASES = [
    (1.0, 0.0, 1.0, -0.4, 2.0, -1.2, 0.8),        # flat surface, singular point inside
    (1.09, 0.24, 1.16, -1.5, 2.5, -1.0, 3.0),      # zx=0.3, zy=0.4, inside
    (1.09, -0.24, 1.16, -1.5, 2.5, -1.0, 3.0),     # B < 0
    (1.25, 0.3, 1.09, -0.7, 1.3, 0.0, 2.0),        # t1 = 0: singular point on the lower edge (l = 1)
    (1.25, 0.3, 1.09, -0.7, 1.3, -2.0, 0.0),       # t2 = 0: singular point on the upper edge (l = M)
    (1.04, -0.12, 1.09, -0.7, 1.3, -5.0, -1.0),    # image box: singular point outside
    (1.0025, 0.01, 1.01, -23.9625, 30.0375, -18.0, 0.0),  # cfg-3-like extents, h = 0.075 offset
    (2.0, 1.5, 1.5625, -0.2, 0.2, -0.2, 0.2),      # steep: zx = 1, zy = 0.75
]


def box(A, B, C, s1, s2, t1, t2):
    f = lambda s, t: 1 / mp.sqrt(A * s * s + B * s * t + C * t * t)
    sb = sorted({mp.mpf(s1), mp.mpf(s2)} | ({mp.mpf(0)} if s1 < 0 < s2 else set()))
    tb = sorted({mp.mpf(t1), mp.mpf(t2)} | ({mp.mpf(0)} if t1 < 0 < t2 else set()))
    return mp.quad(f, sb, tb)


def main():
    out = Path(__file__).with_name("s2_box_integrals.txt")
    with out.open("w") as fh:
        fh.write("# int int ds dt / sqrt(A s^2 + B s t + C t^2); PAPER.md eq.(21) L169, eq.(23) L185-187\n")
        fh.write("# written by tests/golden/make_s2_box_golden.py (mpmath %s, 30 digits)\n" % mp.__version__)
        fh.write("# A B C s1 s2 t1 t2 value\n")
        for c in CASES:
            v = box(*c)
            fh.write(" ".join(repr(float(x)) for x in c) + " " + mp.nstr(v, 22) + "\n")
            print(c, mp.nstr(v, 22))


if __name__ == "__main__":
    main()
