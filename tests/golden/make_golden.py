"""Writes tests/golden/closed_forms.txt from CLOSED FORMS ONLY (no oracle, no CUDA).

The paper prints no numeric worked example, so the stored
values are textbook closed forms of the pair potentials BASELINE.json's north_star names:
  LJ 12-6:  u = 4 eps [(s/r)^12 - (s/r)^6],  F = 24 eps/r [2 (s/r)^12 - (s/r)^6],
            minimum at r* = 2^(1/6) s with u = -eps, u''(r*) = 72 eps / (2^(1/3) s^2)
  reaction field: u = ke q1 q2 (1/r + k r^2 - c), k = (e-1)/((2e+1) rc^3), c = 1/rc + k rc^2,
            u(rc) = 0, F(rc) = ke q1 q2 * 3 / ((2e+1) rc^2)
Run: python tests/golden/make_golden.py
"""
import os
from fractions import Fraction  # noqa: F401  (documents that only exact/closed forms are used)

KE = 138.935458
eps, sig = 0.996, 0.34          # config 1 argon-like LJ
rows = []
rstar = 2.0 ** (1.0 / 6.0) * sig
rows.append(("lj_rstar", rstar))
rows.append(("lj_u_at_rstar", -eps))
rows.append(("lj_upp_at_rstar", 72.0 * eps / (2.0 ** (1.0 / 3.0) * sig * sig)))
for r in (0.30, 0.34, 0.40, 0.55, 0.90):
    x6 = (sig / r) ** 6
    rows.append(("lj_u_r=%.2f" % r, 4.0 * eps * (x6 * x6 - x6)))
    rows.append(("lj_F_r=%.2f" % r, 24.0 * eps / r * (2.0 * x6 * x6 - x6)))
q1, q2, erf, rc = -0.82, 0.41, 78.0, 1.0
k = (erf - 1.0) / ((2.0 * erf + 1.0) * rc ** 3)
c = 1.0 / rc + k * rc * rc
rows.append(("rf_krf_rc3", k * rc ** 3))
rows.append(("rf_F_at_rc", KE * q1 * q2 * 3.0 / ((2.0 * erf + 1.0) * rc * rc)))
for r in (0.25, 0.5, 0.9):
    rows.append(("rf_u_r=%.2f" % r, KE * q1 * q2 * (1.0 / r + k * r * r - c)))
    rows.append(("rf_F_r=%.2f" % r, KE * q1 * q2 * (1.0 / (r * r) - 2.0 * k * r)))
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "closed_forms.txt")
with open(out, "w") as f:
    f.write("# closed-form pair-potential values (see make_golden.py); name value\n")
    for n, v in rows:
        f.write("%s %.17g\n" % (n, v))
print("wrote", out)
