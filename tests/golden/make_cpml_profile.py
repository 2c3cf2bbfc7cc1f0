"""Writes tests/golden/cpml_profile_lo4_hi3.txt -- the pin of the CPML sample POSITIONS (R4 = SURVEY 8(c) O4).

This script calls neither oracle/ nor the CUDA library.  The depth table RHO below is typed by hand from O4's two
sentences, for an axis of n = 12 cells with 4 CPML cells on the low face and 3 on the high face:

    "low slab  rho(u) = (Np - u)/Np        for u < Np,
     high slab rho(u) = (u - (n - Np))/Np  for u > n - Np,  else 0,
     with u = index (E profile, integer position) or index + 1/2 (H profile)"

  low face, Np = 4:   E samples u = 0, 1, 2, 3            -> (4-0)/4, (4-1)/4, (4-2)/4, (4-3)/4   = 1, 3/4, 1/2, 1/4
                      H samples u = 1/2, 3/2, 5/2, 7/2    -> 7/8, 5/8, 3/8, 1/8
  high face, Np = 3:  n - Np = 9.  E samples u = 9, 10, 11 -> 0 (u = 9 is not > 9), 1/3, 2/3
                      H samples u = 19/2, 21/2, 23/2      -> (1/2)/3, (3/2)/3, (5/2)/3            = 1/6, 1/2, 5/6
  the indices 4..8 lie outside both slabs.

The coefficient columns follow from rho by R4's closed forms, evaluated here with Python floats for ONE stated set of
constants (chosen so that every term is switched on: kappa_max != 1, alpha_max != 0):

    m = 3, m_a = 1, kappa_max = 5, alpha_max = 0.05 S/m, sigma_factor = 0.8, eps_r_pml = 4, d = 5 nm, dt = d/(2 c)
    sigma_max = sigma_factor (m+1) / (eta0 d sqrt(eps_r_pml))      =>  sigma_max dt / eps0 = 0.8 * 4 * 0.5 / 2 = 0.8
    sigma = sigma_max rho^m,  kappa = 1 + (kappa_max - 1) rho^m,  alpha = alpha_max (1 - rho)^m_a
    b = exp(-(sigma/kappa + alpha) dt/eps0),   c = sigma (b - 1) / (kappa (sigma + kappa alpha)),   1/kappa

    python tests/golden/make_cpml_profile.py        # rewrites the fixture
"""
import math
import os
from fractions import Fraction as Fr

N, LO, HI = 12, 4, 3
RHO_E = {0: Fr(1), 1: Fr(3, 4), 2: Fr(1, 2), 3: Fr(1, 4), 9: Fr(0), 10: Fr(1, 3), 11: Fr(2, 3)}
RHO_H = {0: Fr(7, 8), 1: Fr(5, 8), 2: Fr(3, 8), 3: Fr(1, 8), 9: Fr(1, 6), 10: Fr(1, 2), 11: Fr(5, 6)}

C0 = 299792458.0
MU0 = 4.0e-7 * math.pi
EPS0 = 1.0 / (MU0 * C0 * C0)
ETA0 = MU0 * C0
M, MA, KMAX, AMAX, SFAC, ERP = 3.0, 1.0, 5.0, 0.05, 0.8, 4.0
D = 5e-9
DT = D / (2.0 * C0)


def coefficients(rho):
    r = float(rho)
    smax = SFAC * (M + 1.0) / (ETA0 * D * math.sqrt(ERP))
    sg, kp, al = smax * r**M, 1.0 + (KMAX - 1.0) * r**M, AMAX * (1.0 - r) ** MA
    b = math.exp(-(sg / kp + al) * DT / EPS0)
    c = 0.0 if sg == 0.0 else sg * (b - 1.0) / (kp * (sg + kp * al))
    return b, c, 1.0 / kp


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cpml_profile_lo4_hi3.txt")
    with open(out, "w") as f:
        f.write("# CPML profile pin (DESIGN.md R4 = SURVEY 8(c) O4; PAPER.md:46 'PML ... on all sides').  Written by\n"
                "# tests/golden/make_cpml_profile.py from a hand-typed depth table; no code of this repo's oracle or CUDA path ran.\n"
                f"# n = {N}  lo = {LO}  hi = {HI}  d = {D!r}  dt = {DT!r}\n"
                f"# cpml = m {M} m_a {MA} kappa_max {KMAX} alpha_max {AMAX} sigma_factor {SFAC} eps_r_pml {ERP}\n"
                "# index | rho_E | bE cE 1/kappaE | rho_H | bH cH 1/kappaH      (slab indices only; 4..8 are interior)\n")
        for u in sorted(RHO_E):
            be, ce, ke = coefficients(RHO_E[u])
            bh, ch, kh = coefficients(RHO_H[u])
            f.write(f"{u} | {RHO_E[u]} | {be!r} {ce!r} {ke!r} | {RHO_H[u]} | {bh!r} {ch!r} {kh!r}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
