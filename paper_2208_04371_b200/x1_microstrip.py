"""The paper's verification case (Fig. 1): a 25-ohm microstrip at the paper's grid size, run on the GPU and
compared with Eq. 7.

    python -m paper_2208_04371_b200.x1_microstrip [--steps 60000] [--device cuda:0]

The line is uniform, so the "tot" run equals the "inc" run: S* = [[0, s], [s, 0]] with s = F[V(y_2)]/F[V(y_1)] (Eq. 1,
Z_r equal at both planes), Z_r = Eq. 2.  Renormalising to 50 ohm (Eq. 5-6) gives S11, S21 to set against Eq. 7 with
Gamma = (Z0 - 50)/(Z0 + 50) and kappa = exp(-j beta l); per-unit-length C = 1/(Z_r v), L = Z_r/v (Eq. 7).
Theory side: Z0,th = 25 ohm (paper); eps_eff from the textbook quasi-static formula the paper's design point follows
(Pozar, ref. [3]): eps_e = (er+1)/2 + (er-1)/2 / sqrt(1 + 12 h/w).
"""
import argparse
import math

import numpy as np

from . import sparams
from .solver import Solver

C0 = 299792458.0


def theory(w):
    t = w["theory"]
    er, u = t["eps_r"], t["w_over_h"]
    ee = (er + 1) / 2 + (er - 1) / 2 / math.sqrt(1 + 12 / u)
    z0_formula = 120 * math.pi / (math.sqrt(ee) * (u + 1.393 + 0.667 * math.log(u + 1.444)))
    return {"eps_eff": ee, "z0_formula": z0_formula, "z0": t["z0"], "gamma": (t["z0"] - 50.0) / (t["z0"] + 50.0)}


def run(w, device="cuda:0", options=None):
    s = Solver.from_workload(w, options=options, device=device)
    s.step(w["steps"])
    (V1, I1), (V2, I2) = s.read_port_dft(0), s.read_port_dft(1)
    impl = s.impl_name
    s.destroy()
    f = np.asarray(w["freqs"])
    l = (w["ports"][1]["ip"] - w["ports"][0]["ip"]) * w["dx"]
    zr = -V1 / I1                                              # oriented along the +x incident wave (R31)
    s21 = V2 / V1                                              # Eq. 1: Z_r is the same at both planes of a uniform line
    zero = np.zeros_like(s21)
    S_star = np.array([[zero, s21], [s21, zero]])
    S = sparams.renormalize(S_star, np.array([zr, zr]))
    theta = -np.unwrap(np.angle(s21))                          # beta l
    beta = theta / l
    v = 2 * np.pi * f / beta
    th = theory(w)
    tl = sparams.telegrapher_from_abcd(sparams.abcd_from_s(S), l, f)   # S -> ABCD -> Z0, L, C (Fig. 1c)
    kappa = np.exp(-1j * 2 * np.pi * f * math.sqrt(th["eps_eff"]) / C0 * l)
    g = th["gamma"]
    return {"freqs": f, "l": l, "impl": impl, "Z_r": zr, "S_star21": s21, "S11": S[0, 0], "S21": S[1, 0],
            "eps_eff": (C0 / v) ** 2, "C": 1.0 / (zr.real * v), "L": zr.real / v,
            "Z0_abcd": tl["Z0"], "C_abcd": tl["C"], "L_abcd": tl["L"], "beta_l": theta,
            "S11_th": (1 - kappa ** 2) * g / (1 - kappa ** 2 * g ** 2), "S21_th": (1 - g ** 2) * kappa / (1 - kappa ** 2 * g ** 2),
            "C_th": math.sqrt(th["eps_eff"]) / (th["z0"] * C0), "L_th": th["z0"] * math.sqrt(th["eps_eff"]) / C0, "theory": th}


def main():
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=60000)
    ap.add_argument("--device", default="cuda:0")
    a = ap.parse_args()
    r = run(W.microstrip_x1(steps=a.steps), a.device)
    print(f"# X1 microstrip, {a.steps} steps, step implementation {r['impl']}, port distance {r['l'] * 1e3:.1f} mm")
    print("# f[GHz]  Re Z_r  Im Z_r  eps_eff  |S11|  |S11_th|  |S21|  |S21_th|  C[pF/m]  L[nH/m]")
    for m in range(0, len(r["freqs"]), 4):
        print(f"{r['freqs'][m] / 1e9:7.2f} {r['Z_r'][m].real:7.3f} {r['Z_r'][m].imag:7.3f} {r['eps_eff'][m]:7.4f} "
              f"{abs(r['S11'][m]):6.4f} {abs(r['S11_th'][m]):6.4f} {abs(r['S21'][m]):6.4f} {abs(r['S21_th'][m]):6.4f} "
              f"{r['C'][m] * 1e12:8.2f} {r['L'][m] * 1e9:8.2f}")
    print(f"# theory: Z0 = {r['theory']['z0']} ohm (formula {r['theory']['z0_formula']:.2f}), eps_eff = {r['theory']['eps_eff']:.4f}, "
          f"C_th = {r['C_th'] * 1e12:.2f} pF/m, L_th = {r['L_th'] * 1e9:.2f} nH/m")


if __name__ == "__main__":
    main()
