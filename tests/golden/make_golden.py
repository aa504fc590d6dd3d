"""Writes the small golden fixtures of tests/golden/ (run from the repo root: python tests/golden/make_golden.py).

weno5_js_example.txt -- the Jiang-Shu WENO5 value (ref 35; eps = 1e-6, exponent 2, reading R7) for
the point values v = (1, 3, 2, 5, 4.5), evaluated in EXACT rational arithmetic (fractions.Fraction) from the
definition, then rounded once to double.  It uses neither oracle/ nor the CUDA path.

wenocu6_beta6_form.txt -- the quadratic form of the six-point Jiang-Shu smoothness measure used by WENO-CU6
(PAPER.md:107 names the scheme, ref 34, and prints no formula; reading R16), derived here in exact rational
arithmetic from its DEFINITION: beta_6 = sum_{l=1..5} dx^(2l-1) int_cell (d^l p/dx^l)^2 dx with p the degree-5 polynomial
whose cell averages over cells i-2..i+3 are f_0..f_5.  Coefficients of f_a f_b (a <= b) times 120960.
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


# ---------------------------------------------------------------------------------------------------------------
# WENO-CU6: quadratic form of beta_6 from its definition
# ---------------------------------------------------------------------------------------------------------------
def _polymul(a, b):
    r = [Fr(0)] * (len(a) + len(b) - 1)
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            r[i + j] += x * y
    return r


def _polyder(a):
    return [a[k] * k for k in range(1, len(a))]


def _polyint(a, lo, hi):
    return sum(c * (hi ** (k + 1) - lo ** (k + 1)) / (k + 1) for k, c in enumerate(a))


n = 6
A = [[_polyint([Fr(0)] * k + [Fr(1)], Fr(2 * (j - 2) - 1, 2), Fr(2 * (j - 2) + 1, 2)) for k in range(n)] for j in range(n)]
M = [row[:] + [Fr(int(i == j)) for j in range(n)] for i, row in enumerate(A)]
for c in range(n):                                    # exact Gauss-Jordan inverse
    piv = next(r for r in range(c, n) if M[r][c] != 0)
    M[c], M[piv] = M[piv], M[c]
    pv = M[c][c]
    M[c] = [x / pv for x in M[c]]
    for r in range(n):
        if r != c and M[r][c] != 0:
            f = M[r][c]
            M[r] = [x - f * y for x, y in zip(M[r], M[c])]
Ainv = [row[n:] for row in M]
P = [[Ainv[k][j] for k in range(n)] for j in range(n)]   # basis polynomial of f_j
lines = ["# beta_6 * 120960 = sum_{a<=b} C[a][b] f_a f_b, f_0..f_5 = cells i-2..i+3; exact, from the definition",
         "# written by tests/golden/make_golden.py"]
for a_ in range(n):
    row = []
    for b_ in range(a_, n):
        pa, pb, acc = P[a_], P[b_], Fr(0)
        for _ in range(1, 6):
            pa, pb = _polyder(pa), _polyder(pb)
            acc += _polyint(_polymul(pa, pb), Fr(-1, 2), Fr(1, 2))
        coef = acc * (1 if a_ == b_ else 2) * 120960
        assert coef.denominator == 1
        row.append(str(coef.numerator))
    lines.append(f"row{a_}=" + ",".join(row))
(Path(__file__).resolve().parent / "wenocu6_beta6_form.txt").write_text("\n".join(lines) + "\n")
print("\n".join(lines))


# ---------------------------------------------------------------------------------------------------------------
# WENO-CU6: beta_6 of a smooth wave at 150 points per wavelength, exact (the case behind reading R16: in doubles the
# value form above loses ~1e-12 of the cell-to-cell difference to cancellation there)
# ---------------------------------------------------------------------------------------------------------------
import math  # noqa: E402

C = [[int(x) for x in ln.split("=")[1].split(",")] for ln in lines if ln.startswith("row")]
out_lines = ["# six doubles v_{i-2}..v_{i+3} (hex) of v(x) = 2 + sin 2 pi x + 0.3 cos 6 pi x at 150 points per unit; beta_6",
             "# (hex, rounded once) from the exact quadratic form of wenocu6_beta6_form.txt evaluated with",
             "# fractions.Fraction on those very doubles; written by tests/golden/make_golden.py"]
for j0 in range(0, 150, 19):
    vs = [2.0 + math.sin(2 * math.pi * (j0 + m) / 150) + 0.3 * math.cos(6 * math.pi * (j0 + m) / 150) for m in range(6)]
    f = [Fr(x) for x in vs]
    b6 = sum(C[a_][k] * f[a_] * f[a_ + k] for a_ in range(6) for k in range(6 - a_)) / 120960
    out_lines.append(",".join(x.hex() for x in vs) + ";" + float(b6).hex())
(Path(__file__).resolve().parent / "wenocu6_beta6_smooth.txt").write_text("\n".join(out_lines) + "\n")
print("\n".join(out_lines))


# ---------------------------------------------------------------------------------------------------------------
# WENO7 (PAPER.md:107 names the scheme, ref 36, and prints no formula; reading R18): candidates, linear
# weights and smoothness indicators derived in exact rational arithmetic from their definitions --
#   candidate k (k = 0..3): the cubic whose cell averages over cells i-3+k .. i+k are the data, evaluated at x_{i+1/2};
#   linear weights d_k: the combination that reproduces the 7-point (degree-6) interpolation;
#   beta_k = sum_{l=1..3} dx^(2l-1) int_cell_i (d^l p_k/dx^l)^2 dx  (the Jiang-Shu measure), as a quadratic form of the
#   four values and of the three first differences D_m = f_{k+m+1} - f_{k+m} of the sub-stencil, both times 240.
# ---------------------------------------------------------------------------------------------------------------
def _basis(cells):
    m = len(cells)
    Am = [[_polyint([Fr(0)] * k + [Fr(1)], Fr(2 * c - 1, 2), Fr(2 * c + 1, 2)) for k in range(m)] for c in cells]
    Mm = [row[:] + [Fr(int(i == j)) for j in range(m)] for i, row in enumerate(Am)]
    for c in range(m):
        piv = next(r for r in range(c, m) if Mm[r][c] != 0)
        Mm[c], Mm[piv] = Mm[piv], Mm[c]
        pv = Mm[c][c]
        Mm[c] = [x / pv for x in Mm[c]]
        for r in range(m):
            if r != c and Mm[r][c] != 0:
                f = Mm[r][c]
                Mm[r] = [x - f * y for x, y in zip(Mm[r], Mm[c])]
    inv = [row[m:] for row in Mm]
    return [[inv[k][j] for k in range(m)] for j in range(m)]


def _polyval(a, x):
    return sum(c * x ** k for k, c in enumerate(a))


w7 = ["# WENO7: exact coefficients from the definitions; written by tests/golden/make_golden.py"]
cands, full = [], [_polyval(p, Fr(1, 2)) for p in _basis(list(range(-3, 4)))]
w7.append("interp7_times_420=" + ",".join(str(x * 420) for x in full))
for k in range(4):
    P4 = _basis(list(range(k - 3, k + 1)))
    cands.append([_polyval(p, Fr(1, 2)) for p in P4])
    w7.append(f"cand{k}_times_12=" + ",".join(str(x * 12) for x in cands[k]))
    B = [[Fr(0)] * 4 for _ in range(4)]
    for a_ in range(4):
        for b_ in range(4):
            pa, pb = P4[a_], P4[b_]
            for _ in range(1, 4):
                pa, pb = _polyder(pa), _polyder(pb)
                B[a_][b_] += _polyint(_polymul(pa, pb), Fr(-1, 2), Fr(1, 2))
    assert all(sum(row) == 0 for row in B)                 # translation invariance
    w7.append(f"beta{k}_values_times_240=" + ";".join(
        ",".join(str(B[a_][b_] * (1 if a_ == b_ else 2) * 240) for b_ in range(a_, 4)) for a_ in range(4)))
    G = [[sum(B[a_][b_] for a_ in range(m + 1, 4) for b_ in range(l + 1, 4)) for l in range(3)] for m in range(3)]
    w7.append(f"beta{k}_differences_times_240=" + ";".join(
        ",".join(str(G[m][l] * (1 if m == l else 2) * 240) for l in range(m, 3)) for m in range(3)))
dlin = [None] * 4
dlin[0] = full[0] / cands[0][0]
dlin[3] = full[6] / cands[3][3]
dlin[1] = (full[1] - dlin[0] * cands[0][1]) / cands[1][0]
dlin[2] = (full[5] - dlin[3] * cands[3][2]) / cands[2][3]
for j in range(7):
    assert sum(dlin[k] * cands[k][j - k] for k in range(4) if 0 <= j - k < 4) == full[j]
w7.append("linear_weights=" + ",".join(str(x) for x in dlin))
(Path(__file__).resolve().parent / "weno7_coefficients.txt").write_text("\n".join(w7) + "\n")
print("\n".join(w7))
