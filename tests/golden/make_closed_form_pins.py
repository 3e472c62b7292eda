"""Writes tests/golden/closed_form_pins.txt: closed-form values (30 digits, mpmath) of the DISCRETE
method on linear flows, used to pin the oracle.  Calls neither the oracle nor the CUDA path.

Derivation (SURVEY.md 8.2 pins P4-P6; PAPER.md:85 RK4, Eq. 1.1, PAPER.md:25 FTLE):
classical RK4 on x' = A x gives x_{n+1} = P(hA) x_n with P(z) = 1 + z + z^2/2 + z^3/6 + z^4/24, and
central differences are exact on a linear map, so G = P(hA)^N, C = G^T G, FTLE = ln(lambda_max(C))/(2T).
  P4 pure strain A = diag(s,-s):   FTLE = ln P(hs) / h;  lambda_max = P(hs)^(2N)
  P5 simple shear u = (gamma y, 0): G = [[1,k],[0,1]], k = gamma T (A nilpotent, RK4 exact);
                                    lambda_max = 1 + k^2/2 + k sqrt(1 + k^2/4)
  P6 rigid rotation u = w(-y, x):   G = |P(i h w)|^N R, FTLE = ln|P(i h w)| / h
"""
import os
from mpmath import mp, mpf, mpc, log, sqrt, pi, fabs

mp.dps = 40
P = lambda z: 1 + z + z**2 / 2 + z**3 / 6 + z**4 / 24
rows = []
for s, h in [(mpf(1), mpf("0.1")), (mpf("0.5"), mpf("0.1")), (mpf(1), mpf("0.05"))]:
    rows.append(("P4_strain_ftle s=%s h=%s" % (s, h), log(P(h * s)) / h))
rows.append(("P4_strain_lambda_max s=1 h=0.1 T=10", P(mpf("0.1")) ** 200))
for g, T in [(mpf("0.5"), mpf(10)), (mpf(1), mpf(10))]:
    k = g * T
    lam = 1 + k**2 / 2 + k * sqrt(1 + k**2 / 4)
    rows.append(("P5_shear_lambda_max gamma=%s T=%s" % (g, T), lam))
    rows.append(("P5_shear_ftle gamma=%s T=%s" % (g, T), log(lam) / (2 * T)))
for name, w, h in [("1", mpf(1), mpf("0.1")), ("2pi/10", 2 * pi / 10, mpf("0.1"))]:
    rows.append(("P6_rotation_ftle omega=%s h=%s" % (name, h), log(fabs(P(mpc(0, h * w)))) / h))
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "closed_form_pins.txt")
with open(out, "w") as f:
    f.write("# closed-form pins of the discrete method (mpmath, 30 digits); see make_closed_form_pins.py\n")
    f.write("# cites: PAPER.md:85 (RK4), PAPER.md:27 (Eq. 1.1), PAPER.md:25 (FTLE); SURVEY.md 8.2 P4-P6\n")
    for k, v in rows:
        f.write("%s | %s\n" % (k, mp.nstr(v, 30)))
print(open(out).read())
