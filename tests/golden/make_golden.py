"""Writes the small golden fixtures of tests/golden/ (run from the repo root: python tests/golden/make_golden.py).

weno5_js_example.txt -- the Jiang-Shu WENO5 value (ref 35; eps = 1e-6, exponent 2, reading R7) for
the point values v = (1, 3, 2, 5, 4.5), evaluated in EXACT rational arithmetic (fractions.Fraction) from the
definition, then rounded once to double.  It uses neither oracle/ nor the CUDA path.
"""
from fractions import Fraction as Fr
from pathlib import Path

v = [Fr(1), Fr(3), Fr(2), Fr(5), Fr(9, 2)]
q = [(2 * v[0] - 7 * v[1] + 11 * v[2]) / 6, (-v[1] + 5 * v[2] + 2 * v[3]) / 6, (2 * v[2] + 5 * v[3] - v[4]) / 6]
b = [Fr(13, 12) * (v[0] - 2 * v[1] + v[2]) ** 2 + Fr(1, 4) * (v[0] - 4 * v[1] + 3 * v[2]) ** 2,
     Fr(13, 12) * (v[1] - 2 * v[2] + v[3]) ** 2 + Fr(1, 4) * (v[1] - v[3]) ** 2,
     Fr(13, 12) * (v[2] - 2 * v[3] + v[4]) ** 2 + Fr(1, 4) * (3 * v[2] - 4 * v[3] + v[4]) ** 2]
eps = Fr(1, 10 ** 6)
d = [Fr(1, 10), Fr(6, 10), Fr(3, 10)]
a = [d[k] / (eps + b[k]) ** 2 for k in range(3)]
val = sum(a[k] * q[k] for k in range(3)) / sum(a)
out = Path(__file__).resolve().parent / "weno5_js_example.txt"
out.write_text(
    "# WENO5-JS (Jiang & Shu; PAPER.md:107 ref 35; eps=1e-6, p=2) at +1/2 for v=(1,3,2,5,4.5); exact rational\n"
    "# arithmetic, written by tests/golden/make_golden.py\n"
    f"v=1,3,2,5,4.5\nvalue={float(val)!r}\nvalue_exact={val.numerator}/{val.denominator}\n")
print(float(val))
