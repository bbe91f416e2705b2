"""Writes tests/golden/boys.txt: Boys function F_m(T) = Gamma(m+1/2) P(m+1/2, T) / (2 T^{m+1/2})
(closed form of eq. 18) evaluated with mpmath at 40 digits.  Calls no repo code."""
import os
import mpmath

mpmath.mp.dps = 40
rows = ["# m  T  F_m(T)   (mpmath 40 digits; definition PAPER.md line 137, eq. 18)"]
for T in ["0.5", "3.0", "12.5", "24.0", "26.0", "40.0", "100.0"]:
    for m in (0, 3, 8, 12):
        t = mpmath.mpf(T)
        v = mpmath.gammainc(m + mpmath.mpf(1) / 2, 0, t) / (2 * t ** (m + mpmath.mpf(1) / 2))
        rows.append(f"{m} {T} {mpmath.nstr(v, 30)}")
open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "boys.txt"), "w").write("\n".join(rows) + "\n")
