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

# ---- harmonic bond and harmonic angle (PAPER.md:40 F = -grad U), textbook closed forms:
#   bond   U = kb/2 (r - b0)^2, |F| = kb |r - b0| along the bond (attractive for r > b0),
#          curvature along the bond u'' = kb, transverse u'/r = kb (1 - b0/r)
#   angle  U = kt/2 (theta - theta0)^2; with a = r_i - r_j along x and b = r_k - r_j in the x-y plane at angle theta:
#          F_i = kt (theta - theta0)/|a| n_i,  n_i = (0, 1, 0)                  (unit, perpendicular to a, towards b)
#          F_k = kt (theta - theta0)/|b| n_k,  n_k = (sin theta, -cos theta, 0) (unit, perpendicular to b, towards a)
#          F_j = -F_i - F_k   (theta > theta0 closes the angle, theta < theta0 opens it)
import math
kb, b0, r = 1.0e5, 0.125, 0.140625          # all exactly representable in FP32 (the topology arrays are FP32)
rows.append(("bond_U", 0.5 * kb * (r - b0) ** 2))
rows.append(("bond_F", kb * (r - b0)))
rows.append(("bond_kpar", kb))
rows.append(("bond_kperp", kb * (1.0 - b0 / r)))
kt, t0, la, lb = 383.0, 1.875, 0.1, 0.15          # theta0 = 1.875 rad (107.43 deg), exact in FP32
for deg in (90, 150):
    th = math.radians(deg)
    dth = th - t0
    rows.append(("angle%d_U" % deg, 0.5 * kt * dth * dth))
    fi = kt * dth / la
    fk = kt * dth / lb
    Fi = (0.0, fi, 0.0)
    Fk = (fk * math.sin(th), -fk * math.cos(th), 0.0)
    for nm, v in (("Fi", Fi), ("Fk", Fk), ("Fj", tuple(-a - b for a, b in zip(Fi, Fk)))):
        for ax, comp in zip("xyz", v):
            rows.append(("angle%d_%s%s" % (deg, nm, ax), comp))

out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "closed_forms.txt")
with open(out, "w") as f:
    f.write("# closed-form pair-potential values (see make_golden.py); name value\n")
    for n, v in rows:
        f.write("%s %.17g\n" % (n, v))
print("wrote", out)
