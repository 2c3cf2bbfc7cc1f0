"""Eq. 5-6 renormalisation to 50 ohm and Eq. 8 phase delay: pins of the oracle's restatement
(oracle/renorm.py) against what the paper and circuit theory fix, then the package's vectorised version against it.

Pins (each fails for a plausible mistake: a missing conjugate, B read as printed (= identity), A and conj A swapped,
the printed numerator (1 - kappa^2) kappa of S21):
  * Z_r = 50 ohm at every port leaves S* unchanged;
  * one port, load Z_L seen from a complex reference Z_r: power-wave S* = (Z_L - conj Z_r)/(Z_L + Z_r) must become the
    ordinary reflection coefficient (Z_L - 50)/(Z_L + 50);
  * a lossless line of impedance 25 ohm, matched in itself (S* = [[0, k], [k, 0]], Z_r = 25): Eq. 7, PAPER.md:97-108,
    with Gamma = -0.333 as printed (tests/golden/paper_values.txt);
  * a two-port built from circuit theory (series impedance between two different complex reference impedances).
"""
import cmath
import math

import numpy as np

from oracle import renorm as R
from paper_2208_04371_b200 import sparams as P


def test_identity_at_50_ohm():
    S = [[0.1 + 0.2j, 0.5 - 0.3j], [0.4 + 0.1j, -0.2 + 0.05j]]
    out = R.renormalize_one(S, [50 + 0j, 50 + 0j])
    assert max(abs(out[i][j] - S[i][j]) for i in range(2) for j in range(2)) < 1e-15


def test_one_port_load():
    for ZL, Zr in ((30 + 12j, 81 + 7j), (75 - 20j, 20 + 5j), (5 + 0j, 25 - 40j)):
        s_star = (ZL - Zr.conjugate()) / (ZL + Zr)
        out = R.renormalize_one([[s_star]], [Zr])
        assert abs(out[0][0] - (ZL - 50) / (ZL + 50)) < 1e-15


def test_eq7_matched_25_ohm_line(golden_dir):
    from tests.test_oracle_pins import load_golden
    g = load_golden(golden_dir)
    gamma_printed, z0 = float(g["gamma_25_50"]), float(g["z0_microstrip_ohm"])
    G = (z0 - 50.0) / (z0 + 50.0)
    assert abs(G - gamma_printed) < 5e-4
    for bl in (0.3, 1.7, 2.9, 5.1):
        k = cmath.exp(-1j * bl)                              # e^{-j beta l}: R30 (this library's DFT sign)
        out = R.renormalize_one([[0, k], [k, 0]], [z0 + 0j, z0 + 0j])
        s11 = (1 - k * k) * G / (1 - k * k * G * G)          # Eq. 7, as printed
        s21 = (1 - G * G) * k / (1 - k * k * G * G)          # Eq. 7 with the numerator read as (1 - Gamma^2) kappa (R30)
        assert abs(out[0][0] - s11) < 1e-15 and abs(out[1][1] - s11) < 1e-15
        assert abs(out[1][0] - s21) < 1e-15 and abs(out[0][1] - s21) < 1e-15
        printed = (1 - k * k) * k / (1 - k * k * G * G)
        assert abs(out[1][0] - printed) > 0.1                # the printed numerator is not what the procedure gives
        # lossless and reciprocal: |S11|^2 + |S21|^2 = 1
        assert abs(abs(out[0][0]) ** 2 + abs(out[1][0]) ** 2 - 1) < 1e-14


def _series_z_two_port(Zs, Z1, Z2):
    """Power-wave S of a series impedance Zs between ports with (complex) reference impedances Z1, Z2, from circuit theory:
    port 1 sees Zs + Z2 when port 2 is terminated in its reference, etc."""
    s11 = (Zs + Z2 - Z1.conjugate()) / (Zs + Z2 + Z1)
    s22 = (Zs + Z1 - Z2.conjugate()) / (Zs + Z1 + Z2)
    s21 = 2 * math.sqrt(Z1.real * Z2.real) / (Zs + Z1 + Z2)
    return [[s11, s21], [s21, s22]]


def test_series_impedance_between_complex_references():
    Zs = 17 - 9j
    for Z1, Z2 in ((30 + 10j, 80 - 25j), (12 - 3j, 50 + 0j)):
        out = R.renormalize_one(_series_z_two_port(Zs, Z1, Z2), [Z1, Z2])
        want = _series_z_two_port(Zs, 50 + 0j, 50 + 0j)
        assert max(abs(out[i][j] - want[i][j]) for i in range(2) for j in range(2)) < 1e-14


def test_phase_delay_of_a_pure_delay():
    f = [1e9 + m * 4e9 for m in range(125)]
    t0 = 3.1e-11                                             # 15 turns of phase over the band: unwrapping is exercised
    s = [0.8 * cmath.exp(-2j * math.pi * fm * t0) for fm in f]
    tau = R.phase_delay(s, f)
    assert max(abs(t + t0) for t in tau) < 1e-22 + 1e-12 * t0
    th = R.unwrapped_phase_deg(s)
    assert all(b < a for a, b in zip(th, th[1:])) and th[-1] < -5000


def test_package_matches_oracle_restatement():
    r = np.random.default_rng(5)
    N, F = 4, 9
    S = (r.normal(size=(N, N, F)) + 1j * r.normal(size=(N, N, F))) * 0.4
    Z = r.uniform(10, 120, size=(N, F)) + 1j * r.normal(size=(N, F)) * 20
    a = np.array(R.renormalize(S.tolist(), Z.tolist()))
    assert np.abs(a - P.renormalize(S, Z)).max() < 1e-13
    f = np.linspace(1e9, 5e11, 64)
    s = np.exp(-1j * 2 * np.pi * f * 3e-11) * 0.7
    assert np.abs(np.array(R.phase_delay(s.tolist(), f.tolist())) - P.phase_delay(s, f)).max() < 1e-20


def test_drive_port_moves_the_source():
    import workloads as W
    w = W.interconnect_c4(run="inc", div=8, steps=10, npml=5, nf=4)
    for j, want_dir in ((0, 1), (1, -1), (2, 1), (3, -1)):
        wj, d = W.drive_port(w, j)
        assert d == want_dir
        assert [q["has_source"] for q in wj["ports"]] == [int(q == j) for q in range(4)]
        t = wj["ports"][j]
        assert (t["sj0"], t["sj1"], t["sk0"], t["sk1"]) == (t["vj0"], t["vj1"], t["vk0"], t["vk1"])
        assert (t["ip"] - t["is"]) * d == abs(w["ports"][0]["ip"] - w["ports"][0]["is"])
    assert w["ports"][0]["has_source"] == 1                  # the input workload is not modified


def test_abcd_and_telegrapher_recover_a_lossy_line():
    """PAPER.md:89 (S* -> ABCD -> characteristic impedance and RLGC of the simplest Telegrapher's model): a uniform lossy
    line built from R, L, G, C by textbook circuit theory must come back, through several turns of phase."""
    R_, L_, G_, C_ = 120.0, 2.5e-7, 0.02, 1.0e-10
    l = 0.05
    f = np.linspace(0.2e9, 20e9, 400)
    w = 2 * np.pi * f
    z = R_ + 1j * w * L_
    y = G_ + 1j * w * C_
    gamma, zc = np.sqrt(z * y), np.sqrt(z / y)
    A = np.cosh(gamma * l); B = zc * np.sinh(gamma * l); Cm = np.sinh(gamma * l) / zc
    # S on 50 ohm from ABCD (textbook), then back through the package
    den = A + B / 50 + Cm * 50 + A
    S = np.array([[(A + B / 50 - Cm * 50 - A) / den, 2 * (A * A - B * Cm) / den], [2 / den, (-A + B / 50 - Cm * 50 + A) / den]])
    abcd = P.abcd_from_s(S)
    assert np.abs(abcd[0, 0] - A).max() < 1e-9 and np.abs(abcd[0, 1] - B).max() < 1e-7 and np.abs(abcd[1, 0] - Cm).max() < 1e-11
    t = P.telegrapher_from_abcd(abcd, l, f)
    assert np.abs(t["Z0"] / zc - 1).max() < 1e-9
    assert np.abs(t["R"] / R_ - 1).max() < 1e-6 and np.abs(t["L"] / L_ - 1).max() < 1e-8
    assert np.abs(t["G"] / G_ - 1).max() < 1e-6 and np.abs(t["C"] / C_ - 1).max() < 1e-8
    assert (np.diff(t["gamma"].imag) > 0).all() and t["gamma"].imag[-1] * l > 4 * np.pi      # unwrapped past 2 turns
