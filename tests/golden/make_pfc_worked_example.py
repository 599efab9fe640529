"""Writes pfc_worked_example.txt: an 8-cell worked example of the 1D PFC remap (limiters on, f_inf = 1,
periodic, uniform shift).  The paper (arXiv 1406.5445) prints no worked example; these values are the
exact rational evaluation of its eq. (17) with the reconstruction of eqs. (40), (43)-(45) (sign of
erratum R4), rounded to double.  Calls neither oracle/ nor the CUDA path.

    python tests/golden/make_pfc_worked_example.py
"""
import os
import sys
from fractions import Fraction

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
from pfc_exact import exact_remap_periodic  # noqa: E402

f = [Fraction(v) for v in ("0", "0", "1/10", "1", "9/10", "1/5", "0", "0")]
shifts = [Fraction(1, 4), Fraction(-3, 5), Fraction(3, 2), Fraction(-23, 10)]
with open(os.path.join(HERE, "pfc_worked_example.txt"), "w") as fh:
    fh.write("# 1D PFC remap worked example; PAPER.md eqs. 17, 38, 40, 43-47 (not printed by the paper;\n")
    fh.write("# exact rational integration, see make_pfc_worked_example.py).  Row: shift sigma, then f'_0..f'_7\n")
    fh.write("f " + " ".join(repr(float(v)) for v in f) + "\n")
    for s in shifts:
        out = exact_remap_periodic(f, [s] * 9, Fraction(1), 1)
        fh.write(repr(float(s)) + " " + " ".join(repr(float(v)) for v in out) + "\n")
