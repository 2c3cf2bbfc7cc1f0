"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Each test names the pin id of DESIGN.md / SURVEY.md 8(c)-P and the passage it rests on.  A plausible
mistake anywhere in oracle/yee_oracle.cpp (dropped term, wrong sign or index, transposed operand,
wrong time stamp) fails at least one of them.
"""
import math
from fractions import Fraction
import os

import numpy as np
import pytest

import workloads as W
from oracle import sparams as osp
from oracle import yee
from oracle.yee import EX, EY, EZ, HX, HY, HZ, YeeOracle

from .ref_numpy import NumpyYee

C0 = 299792458.0
MU0 = 4e-7 * math.pi
EPS0 = 1 / (MU0 * C0**2)
ETA0 = MU0 * C0


# ------------------------------------------------------------------------------------------------
def load_golden(golden_dir):
    out = {}
    with open(os.path.join(golden_dir, "paper_values.txt")) as f:
        for line in f:
            if line.startswith("#") or "=" not in line:
                continue
            key, rest = line.split("=", 1)
            val = rest.split("|")[0].strip()
            out[key.strip()] = val
    return out


def test_constants_R2():
    c, mu0, eps0, eta0 = yee.constants()
    assert c == 299792458.0
    assert abs(mu0 - 4e-7 * math.pi) < 1e-21
    assert abs(eps0 * mu0 * c * c - 1) < 1e-15
    assert abs(eta0 - 376.730313) < 1e-5


def test_P1_cfl_values_printed_in_the_paper(golden_dir):
    g = load_golden(golden_dir)
    # 200x1000x50 cells, h = 1 mm = 10 cells -> d = 0.1 mm, CFL number 0.9
    assert 0.9 * yee.cfl_dt(1e-4, 1e-4, 1e-4) == pytest.approx(float(g["dt_microstrip_s"]), rel=2e-3)
    # (20, 50, 5) nm, CFL number 0.9
    assert 0.9 * yee.cfl_dt(20e-9, 50e-9, 5e-9) == pytest.approx(float(g["dt_cmos_s"]), rel=2e-3)
    # bookkeeping of PAPER.md:114-116
    assert [200 * 20e-3, 120 * 50e-3, 800 * 5e-3] == pytest.approx([float(v) for v in g["cmos_domain_um"].split()])
    # record length -> lowest resolved frequency
    assert 1 / (60000 * 0.9 * yee.cfl_dt(1e-4, 1e-4, 1e-4)) == pytest.approx(float(g["fmin_microstrip_hz"]), rel=5e-2)
    assert 1 / (1.4e6 * 0.9 * yee.cfl_dt(20e-9, 50e-9, 5e-9)) == pytest.approx(float(g["fmin_cmos_hz"]), rel=5e-2)


def test_P1_create_rejects_dt_above_cfl():
    d = 5e-9
    lim = yee.cfl_dt(d, d, d)
    YeeOracle(4, 4, 4, d, d, d, lim * 0.999999)
    with pytest.raises(ValueError):
        YeeOracle(4, 4, 4, d, d, d, lim * 1.000001)
    with pytest.raises(ValueError):
        YeeOracle(1, 4, 4, d, d, d, lim * 0.5)


def _spectrum(kind, sigma, freqs, f0=0.0):
    t0 = 3 * sigma
    t = np.linspace(0, 12 * sigma, 24001)
    g = yee.waveform(kind, t, t0, sigma, f0)
    ph = np.exp(-2j * np.pi * np.outer(freqs, t))
    return np.abs(np.trapezoid(ph * g, t, axis=1))


@pytest.mark.parametrize("sigma,key", [(11.254e-12, "fp_sigma_11.254ps_hz"), (10.146e-15, "fp_sigma_10.146fs_hz"),
                                       (1.45e-15, "fp_sigma_1.45fs_hz")])
def test_T3_eq3_peak_frequency(golden_dir, sigma, key):
    """Eq. 3 with f_p = (sqrt(2) pi sigma)^-1: pins exp(-u^2), not exp(-u^2/2)."""
    g = load_golden(golden_dir)
    fp = float(g[key])
    f = np.linspace(0.5 * fp, 1.5 * fp, 2001)
    s = _spectrum(yee.W_DGAUSS, sigma, f)
    assert f[np.argmax(s)] == pytest.approx(fp, rel=3e-3)
    assert f[np.argmax(s)] == pytest.approx(1 / (math.sqrt(2) * math.pi * sigma), rel=1e-3)


@pytest.mark.parametrize("sigma,lo,hi", [(10.146e-15, "drop3_lo_10.146fs_hz", "drop3_hi_10.146fs_hz"),
                                         (1.45e-15, "drop3_lo_1.45fs_hz", "drop3_hi_1.45fs_hz")])
def test_T4_eq3_three_orders_of_magnitude(golden_dir, sigma, lo, hi):
    """the spectrum of Eq. 3 is down 'three orders' at the quoted band edges."""
    g = load_golden(golden_dir)
    fp = 1 / (math.sqrt(2) * math.pi * sigma)
    s = _spectrum(yee.W_DGAUSS, sigma, np.array([fp, float(g[lo]), float(g[hi])]))
    for v in s[1:] / s[0]:
        assert 10 ** -3.7 < v < 10 ** -2.5   # "three orders", read to +-0.7 of an order


def test_waveforms_R6_values():
    s = 2.0
    # GAUSS at t0 +- sigma is 1/e; DGAUSS is odd about t0 with extremum at u = 1/sqrt(2)
    assert yee.waveform(yee.W_GAUSS, [6.0, 8.0, 4.0], 6.0, s)[0] == 1.0
    assert yee.waveform(yee.W_GAUSS, [8.0], 6.0, s)[0] == pytest.approx(math.exp(-1))
    d = yee.waveform(yee.W_DGAUSS, [6 - s / math.sqrt(2), 6.0, 6 + s / math.sqrt(2)], 6.0, s)
    assert d[1] == 0 and d[0] == pytest.approx(-d[2]) and d[0] == pytest.approx(math.sqrt(2) * math.exp(-0.5))
    gs = yee.waveform(yee.W_GSINE, [6.0 + 0.25 / 3.0], 6.0, 1e9, 3.0)  # quarter period of f0 = 3, huge sigma
    assert gs[0] == pytest.approx(1.0, abs=1e-12)


# ------------------------------------------------------------------------------------------------
# P2  exact discrete eigenmode + Yee dispersion relation
# ------------------------------------------------------------------------------------------------
def _eigenmode(nx, ny, nz, dx, dy, dz, m, pol):
    k_, j_, i_ = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    kx, ky, kz = (m[a] * np.pi / (n * d) for a, (n, d) in enumerate([(nx, dx), (ny, dy), (nz, dz)]))
    K = np.array([2 / d * np.sin(k * d / 2) for k, d in [(kx, dx), (ky, dy), (kz, dz)]])
    A = np.cross(K, pol)                      # A perpendicular to K: discrete divergence-free
    sx, cx = np.sin(kx * i_ * dx), np.cos(kx * (i_ + .5) * dx)
    sy, cy = np.sin(ky * j_ * dy), np.cos(ky * (j_ + .5) * dy)
    sz, cz = np.sin(kz * k_ * dz), np.cos(kz * (k_ + .5) * dz)
    E = [A[0] * cx * sy * sz, A[1] * sx * cy * sz, A[2] * sx * sy * cz]
    KxA = np.cross(K, A)                      # discrete curl of E at the H sample points
    curlE = [KxA[0] * sx * cy * cz, KxA[1] * cx * sy * cz, KxA[2] * cx * cy * sz]
    return K, A, E, curlE


@pytest.mark.parametrize("m", [(1, 2, 1), (0, 1, 1), (2, 1, 3)])
def test_P2_exact_discrete_eigenmode_and_dispersion(m):
    nx, ny, nz, dx, dy, dz = 8, 6, 10, 5e-9, 4e-9, 6e-9
    dt = 0.9 * yee.cfl_dt(dx, dy, dz)
    K, A, E, curlE = _eigenmode(nx, ny, nz, dx, dy, dz, m, [0.3, -1.0, 0.7])
    o = YeeOracle(nx, ny, nz, dx, dy, dz, dt)
    o.set_boundary([0] * 6)
    o.commit()
    for c in range(3):
        o.write_field(c, E[c])
        o.write_field(3 + c, dt / (2 * MU0) * curlE[c])     # H^{-1/2} = -H^{+1/2}
    # Yee numerical dispersion: sin(w dt/2) = (c dt/2) |K|
    w = 2 / dt * math.asin(C0 * dt / 2 * np.linalg.norm(K))
    err = 0.0
    for n in range(1, 401):
        o.step(1)
        if n % 7 == 0 or n == 400:
            for c in range(3):
                err = max(err, np.abs(o.read_field(c) - E[c] * math.cos(w * n * dt)).max())
    assert err / np.abs(A).max() < 1e-12


def test_P2_transposed_operand_would_fail():
    """The pin discriminates: the same mode with kx and ky swapped in the reference is far off."""
    nx, ny, nz, dx, dy, dz = 8, 6, 10, 5e-9, 4e-9, 6e-9
    dt = 0.9 * yee.cfl_dt(dx, dy, dz)
    K, A, E, curlE = _eigenmode(nx, ny, nz, dx, dy, dz, (1, 2, 1), [0.3, -1.0, 0.7])
    o = YeeOracle(nx, ny, nz, dx, dy, dz, dt)
    o.set_boundary([0] * 6)
    o.commit()
    for c in range(3):
        o.write_field(c, E[c])
        o.write_field(3 + c, dt / (2 * MU0) * curlE[c])
    o.step(50)
    w_wrong = C0 * math.sqrt(sum((mm * math.pi / (n * d)) ** 2 for mm, n, d in [(2, nx, dx), (1, ny, dy), (1, nz, dz)]))
    assert np.abs(o.read_field(EZ) - E[2] * math.cos(w_wrong * 50 * dt)).max() / np.abs(A).max() > 1e-2


# ------------------------------------------------------------------------------------------------
# P3  leapfrog energy invariant
# ------------------------------------------------------------------------------------------------
def test_P3_leapfrog_energy_invariant():
    nx, ny, nz, dx, dy, dz = 9, 7, 8, 5e-9, 7e-9, 4e-9
    dt = 0.99 * yee.cfl_dt(dx, dy, dz)
    r = np.random.default_rng(3)
    o = YeeOracle(nx, ny, nz, dx, dy, dz, dt)
    o.set_boundary([0] * 6)
    o.commit()
    E = [r.standard_normal((nz, ny, nx)) for _ in range(3)]
    E[0][0] = 0; E[0][:, 0] = 0
    E[1][0] = 0; E[1][:, :, 0] = 0
    E[2][:, 0] = 0; E[2][:, :, 0] = 0
    H = [r.standard_normal((nz, ny, nx)) / ETA0 for _ in range(3)]
    H[0][:, :, 0] = 0; H[1][:, 0] = 0; H[2][0] = 0      # normal H on the low walls
    for c in range(3):
        o.write_field(c, E[c])
        o.write_field(3 + c, H[c])
    Ws = []
    Hm = [o.read_field(3 + c) for c in range(3)]
    for n in range(300):
        En = [o.read_field(c) for c in range(3)]
        o.step(1)
        Hp = [o.read_field(3 + c) for c in range(3)]
        Ws.append(0.5 * EPS0 * sum((e * e).sum() for e in En) + 0.5 * MU0 * sum((a * b).sum() for a, b in zip(Hp, Hm)))
        Hm = Hp
    Ws = np.array(Ws)
    assert np.abs(Ws / Ws[0] - 1).max() < 1e-13
    # the naive 1/2 mu |H^{n+1/2}|^2 form is NOT conserved -- the invariant is specific
    assert Ws[0] > 0


# ------------------------------------------------------------------------------------------------
# P4  lossy / magnetic cavity: scalar three-term recurrence
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("eps_r,sigma,mu_r", [(3.9, 2e4, 1.0), (1.0, 5.8e7, 1.5), (7.0, 0.0, 2.0)])
def test_P4_lossy_cavity_recurrence(eps_r, sigma, mu_r):
    nx, ny, nz, dx, dy, dz = 6, 8, 7, 5e-9, 5e-9, 2.5e-9
    dt = 0.9 * yee.cfl_dt(dx, dy, dz)
    K, A, E, _ = _eigenmode(nx, ny, nz, dx, dy, dz, (1, 1, 2), [1.0, 0.2, -0.4])
    o = YeeOracle(nx, ny, nz, dx, dy, dz, dt)
    o.set_boundary([0] * 6)
    full = lambda v: [np.full((nz, ny, nx), v)] * 3
    o.set_materials_full(full(eps_r), full(sigma), full(mu_r))
    o.commit()
    for c in range(3):
        o.write_field(c, E[c])
    a = sigma * dt / (2 * EPS0 * eps_r)
    Ca, Cb = (1 - a) / (1 + a), dt / (EPS0 * eps_r) / (1 + a)
    q = Cb * dt * float(K @ K) / (MU0 * mu_r)
    s_prev, s = 1.0, Ca - q
    err = 0.0
    for n in range(1, 200):
        o.step(1)
        for c in range(3):
            err = max(err, np.abs(o.read_field(c) - s * E[c]).max())
        s_prev, s = s, (1 + Ca - q) * s - Ca * s_prev
    assert err / np.abs(A).max() < 1e-12


# ------------------------------------------------------------------------------------------------
# C0 / north_star: analytic resonant frequencies of a PEC rectangular cavity
# ------------------------------------------------------------------------------------------------
def test_C0_cavity_resonances_match_analytic_modes():
    w = W.cavity_c0()
    o = YeeOracle.from_workload(w)
    n, d, dt = w["nx"], w["dx"], w["dt"]
    i, j, k = w["source_cell"]
    pi, pj, pk = (i + 5) % (n - 2) + 1, (j + 9) % (n - 2) + 1, (k + 3) % (n - 2) + 1
    hist = []
    for _ in range(w["steps"]):
        o.step(1)
        hist.append(o.read_field(EZ)[pk, pj, pi])
    hist = np.array(hist)
    t = (np.arange(hist.size) + 1) * dt
    start = 120                                          # source has died out by then (t0 + 3 sigma = 72 dt)
    win = np.hanning(hist.size - start)
    f = np.arange(1000e12, 3000e12, 1e12)
    spec = np.abs(np.exp(-2j * np.pi * np.outer(f, t[start:])) @ (hist[start:] * win))
    peaks = [f[q] for q in range(1, f.size - 1) if spec[q] > spec[q - 1] and spec[q] > spec[q + 1]
             and spec[q] > 0.1 * spec.max()]          # Hann side lobes sit at -31 dB = 2.8 %
    a = n * d
    analytic = sorted({round(C0 / 2 * math.sqrt(m1 * m1 + m2 * m2 + m3 * m3) / a / 1e12, 3)
                       for m1 in range(4) for m2 in range(4) for m3 in range(4)
                       if (m1 > 0) + (m2 > 0) + (m3 > 0) >= 2})
    assert analytic[0] == pytest.approx(1324.9, rel=1e-3)         # (1,1,0) of a 160 nm cube
    assert len(peaks) >= 3
    for p in peaks:
        nearest = min(analytic, key=lambda x: abs(x * 1e12 - p))
        assert abs(nearest * 1e12 - p) / p < 0.015, (p, nearest)
    # lowest peak is the (1,1,0) family and it sits at the DISCRETE eigenfrequency (below the analytic one)
    K2 = 2 * (2 / d * math.sin(math.pi / (2 * n))) ** 2
    f110 = math.asin(C0 * dt / 2 * math.sqrt(K2)) / (math.pi * dt)
    assert abs(peaks[0] - f110) / f110 < 0.01
    # energy conservation once the source is off (P3 on the C0 run itself)
    # (W needs H at two times: re-run the last steps)
    Hm = [o.read_field(3 + c) for c in range(3)]
    Ws = []
    for _ in range(20):
        En = [o.read_field(c) for c in range(3)]
        o.step(1)
        Hp = [o.read_field(3 + c) for c in range(3)]
        Ws.append(0.5 * EPS0 * sum((e * e).sum() for e in En) + 0.5 * MU0 * sum((x * y).sum() for x, y in zip(Hp, Hm)))
        Hm = Hp
    Ws = np.array(Ws)
    assert np.abs(Ws / Ws[0] - 1).max() < 1e-12


# ------------------------------------------------------------------------------------------------
# P5 / P6 / S11 pin: vacuum parallel-plate line through the whole V / I / DFT / S* chain
# ------------------------------------------------------------------------------------------------
def _run_pplate(eps_step=None, steps=3000, f32=False, **kw):
    w = W.parallel_plate(steps=steps, **kw)
    if eps_step is not None:
        i0, er = eps_step
        e = [a.copy() for a in w["materials"]["eps_r"]]
        e[0][:, :, i0:] = er                  # Ex(i+1/2) inside the filled half
        for c in (1, 2):                      # tangential Ey, Ez: interface plane gets the mean
            e[c][:, :, i0 + 1:] = er
            e[c][:, :, i0] = 0.5 * (1 + er)
        w["materials"]["eps_r"] = e
    o = YeeOracle.from_workload(w, f32=f32)
    o.step(steps)
    return w, o


def test_P5_P6_parallel_plate_impedance_and_numerical_dispersion():
    fr = np.linspace(2e12, 300e12, 40)
    w, o = _run_pplate(freqs=fr)
    V1, I1 = o.read_port_dft(0)
    V2, I2 = o.read_port_dft(1)
    Z_th = ETA0 * w["gap_m"] / w["width_m"]
    # P5: |V/I| = eta0 d / w at both planes, every frequency
    assert np.abs(np.abs(V1 / I1) / Z_th - 1).max() < 1e-3
    assert np.abs(np.abs(V2 / I2) / Z_th - 1).max() < 1e-3
    # sign convention (R7): a +x travelling wave has Re(V/I) < 0
    assert (np.real(V1 / I1) < 0).all()
    # P6: S*_21 = exp(-j k_num l), k_num from the Yee dispersion relation on the axis
    S = osp.s_star_column(0, [V1, V2], [I1, I2], [V1, V2])
    dx, dt = w["dx"], w["dt"]
    knum = 2 / dx * np.arcsin(np.sin(np.pi * fr * dt) * dx / (C0 * dt))
    L = (w["ports"][1]["ip"] - w["ports"][0]["ip"]) * dx
    S21 = np.array(S[1])
    assert np.abs(S21 - np.exp(-1j * knum * L)).max() < 1e-5
    # ... and the test discriminates: the exact (continuum) k is measurably worse
    assert np.abs(S21 - np.exp(-2j * np.pi * fr / C0 * L)).max() > 2e-5
    # S*_11 of a uniform line is exactly 0 (tot == inc)
    assert np.abs(np.array(S[0])).max() == 0.0


def test_S11_pin_dielectric_step_gives_gamma_minus_one_third(golden_dir):
    """Half of the line filled with eps_r = 4 halves the impedance: Gamma = (Z2-Z1)/(Z2+Z1) = -1/3, the
    same value the paper quotes for its 25-vs-50 ohm mismatch.  Pins Eq. 1's i = j branch
    (V_ref = V_tot - V_inc) and the i != j branch with unequal Z_r (transmission 1 + Gamma)."""
    gamma = float(load_golden(golden_dir)["gamma_25_50"])
    fr = np.linspace(2e12, 20e12, 10)
    kw = dict(nx=400, ip1=100, ip2=300, isrc=60, freqs=fr, sig_dt=40.0)
    _, oi = _run_pplate(steps=6000, **kw)
    _, ot = _run_pplate(eps_step=(200, 4.0), steps=6000, **kw)
    Vi = [oi.read_port_dft(p)[0] for p in (0, 1)]
    Ii = [oi.read_port_dft(p)[1] for p in (0, 1)]
    Vt = [ot.read_port_dft(p)[0] for p in (0, 1)]
    S = osp.s_star_column(0, Vi, Ii, Vt)
    # reference planes: port 1 is 100 cells before the step -> S11 = Gamma * exp(-2 j k l1)
    assert np.abs(np.abs(np.array(S[0])) - abs(gamma)).max() < 5e-3
    k1 = 2 * np.pi * fr / C0
    assert np.abs(np.array(S[0]) * np.exp(2j * k1 * 100 * 5e-9) - gamma).max() < 2e-2
    # Eq. 1 normalises port 2 with the *incident-run* Z_r (equal at both planes), so |S21| = 1 + Gamma
    assert np.abs(np.abs(np.array(S[1])) - (1 + gamma)).max() < 5e-3


# ------------------------------------------------------------------------------------------------
# P7  running DFT against a brute-force transform of the stored history
# ------------------------------------------------------------------------------------------------
def test_P7_running_dft_equals_bruteforce():
    w = W.random_box(11, steps=60)
    o = YeeOracle.from_workload(w)
    V, I = [], []
    for _ in range(60):
        o.step(1)
        v, i = o.read_port_last(1)
        V.append(v)
        I.append(i)
    V, I = np.array(V), np.array(I)
    n = np.arange(60)
    Vh, Ih = o.read_port_dft(1)
    for m, f in enumerate(w["freqs"]):
        bv = sum(V[q] * np.exp(-2j * np.pi * f * (q + 1) * w["dt"]) for q in n) * w["dt"]
        bi = sum(I[q] * np.exp(-2j * np.pi * f * (q + 0.5) * w["dt"]) for q in n) * w["dt"]
        assert abs(Vh[m] - bv) <= 1e-13 * np.abs(V).max() * 60 * w["dt"]
        assert abs(Ih[m] - bi) <= 1e-13 * np.abs(I).max() * 60 * w["dt"]
    assert np.abs(V).max() > 0 and np.abs(I).max() > 0


# ------------------------------------------------------------------------------------------------
# P8  CPML reflection level
# ------------------------------------------------------------------------------------------------
def test_P8_cpml_reflection_below_minus_60_dB():
    steps = 900
    w = W.parallel_plate(nx=160, ip1=40, ip2=120, isrc=30, npml=10, steps=steps)
    wl = W.parallel_plate(nx=640, ip1=40, ip2=120, isrc=30, npml=10, steps=steps)  # end reflection cannot return
    o, ol = YeeOracle.from_workload(w), YeeOracle.from_workload(wl)
    a, b = [], []
    for _ in range(steps):
        o.step(1); ol.step(1)
        a.append(o.read_port_last(1)[0]); b.append(ol.read_port_last(1)[0])
    a, b = np.array(a), np.array(b)
    assert np.abs(b).max() > 0
    assert np.abs(a - b).max() / np.abs(b).max() < 1e-3          # -60 dB
    # a bare PEC wall instead of the CPML reflects everything (the pin discriminates)
    w0 = W.parallel_plate(nx=160, ip1=40, ip2=120, isrc=30, npml=0, steps=steps)
    w0["pml"] = [0] * 6
    o0 = YeeOracle.from_workload(w0)
    c = []
    for _ in range(steps):
        o0.step(1); c.append(o0.read_port_last(1)[0])
    assert np.abs(np.array(c) - b).max() / np.abs(b).max() > 0.5


# ------------------------------------------------------------------------------------------------
# P10  independent whole-array formulation on tiny grids, every term switched on
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,indexed,with_mu,pml", [
    (1, True, True, (3, 4, 2, 3, 0, 3)),
    (2, False, False, (0, 3, 3, 0, 2, 2)),
    (3, True, False, (2, 2, 2, 2, 2, 2)),
    (4, False, True, (0, 0, 0, 0, 0, 0)),
])
def test_P10_oracle_equals_numpy_formulation(seed, indexed, with_mu, pml):
    w = W.random_box(seed, indexed=indexed, with_mu=with_mu, pml=pml, steps=40)
    o = YeeOracle.from_workload(w, track_max=True)
    r = NumpyYee(w)
    o.step(40)
    r.step(40)
    emax, hmax = o.running_max()
    assert emax > 0 and hmax > 0
    # R13: the running maxima are max|E| and max|H| over space and time, two separate scalars (the numpy formulation
    # tracks them itself; fields agree to 1e-12, so do their maxima)
    assert abs(emax / r.emax - 1) < 1e-12 and abs(hmax / r.hmax - 1) < 1e-12
    for c in range(6):
        scale = emax if c < 3 else hmax
        assert np.abs(o.read_field(c) - r.field(c)).max() / scale < 1e-12, c
    for p in range(2):
        V, I = o.read_port_dft(p)
        assert np.abs(V - r.Vhat[p]).max() <= 1e-12 * np.abs(r.Vhat).max()
        assert np.abs(I - r.Ihat[p]).max() <= 1e-12 * np.abs(r.Ihat).max()
    if any(pml):
        assert o.psi_norms().max() > 0


# ------------------------------------------------------------------------------------------------
# R13  the running maximum (denominator of every field tolerance of the GPU parity tests)
# ------------------------------------------------------------------------------------------------
def test_R13_running_max_is_separate_for_E_and_H_over_space_and_time_and_resets_at_commit():
    """A pulse in a lossy box peaks mid-run and decays: "the maximum of the last step", "one maximum over E and H
    together", "a sum" and "never reset at commit" all fail one of the asserts below.  The expected values come from
    the independent numpy formulation's own per-step history."""
    w = W.random_box(7, indexed=False, with_mu=False, pml=(3, 3, 3, 3, 0, 3), steps=160, pec_frac=0.0)
    for c in range(3):                                                   # lossy everywhere: the pulse dies out
        w["materials"]["sigma"][c] = np.maximum(np.where(np.isinf(w["materials"]["sigma"][c]), 0.0,
                                                         w["materials"]["sigma"][c]), 3e5)
    o = YeeOracle.from_workload(w, track_max=True)
    r = NumpyYee(w)
    o.step(160); r.step(160)
    emax, hmax = o.running_max()
    eh, hh = np.array(r.emax_hist), np.array(r.hmax_hist)
    # the case discriminates: the peak lies mid-run, the last step is far below it, |E| and |H| differ by orders
    assert 5 < eh.argmax() < 100 and eh[-1] < 0.2 * eh.max() and hh[-1] < 0.2 * hh.max()
    assert eh.max() > 50 * hh.max()
    assert abs(emax / eh.max() - 1) < 1e-12                             # max over time of max over space of |E| ...
    assert abs(hmax / hh.max() - 1) < 1e-12                             # ... and of |H|, separately
    # and it is the maximum over all three components of the family, not of one of them
    per_comp = [max(np.abs(r.field(c)).max() for c in (0, 1, 2)), max(np.abs(r.field(c)).max() for c in (3, 4, 5))]
    assert per_comp[0] <= emax and per_comp[1] <= hmax
    # without tracking the maxima stay zero (the GPU tests would divide by zero, loudly)
    o2 = YeeOracle.from_workload(w, track_max=False)
    o2.step(5)
    assert o2.running_max() == (0.0, 0.0)
    # a second commit zeroes the maxima with the rest of the state
    o.commit()
    assert o.running_max() == (0.0, 0.0) and o.step_count == 0
    o.step(4)
    e4, h4 = o.running_max()
    assert abs(e4 / eh[:4].max() - 1) < 1e-12 and abs(h4 / hh[:4].max() - 1) < 1e-12


def test_R13_running_max_from_an_initial_state_whose_E_peak_is_at_step_zero():
    """An initial E_z column profile (written through write_field, source off) that only decays afterwards: the E
    maximum is the one of the first steps, the H maximum is reached later, and in SI units |H| is two orders below
    |E|, so one maximum over E and H together (or H scaled by eta0) shows up here.  Expected values: the numpy
    formulation started from the same state."""
    w = W.random_box(8, indexed=False, with_mu=False, pml=(0, 0, 0, 0, 0, 0), steps=6, pec_frac=0.0)
    for c in range(3):
        w["materials"]["sigma"][c] = np.zeros_like(w["materials"]["sigma"][c])
        w["materials"]["eps_r"][c] = np.ones_like(w["materials"]["eps_r"][c])
    w["ports"][0]["amp"] = 0.0
    nz, ny, nx = w["nz"], w["ny"], w["nx"]
    ez0 = np.zeros((nz, ny, nx))
    ez0[:, 1:, 1:] = (1.0 + np.arange(nz))[:, None, None]                # uniform in x, y; rows i = 0, j = 0 are walls
    o = YeeOracle.from_workload(w, track_max=True)
    r = NumpyYee(w)
    o.write_field(EZ, ez0)
    r.E["z"] = ez0.copy()
    o.step(6); r.step(6)
    emax, hmax = o.running_max()
    assert abs(emax / r.emax - 1) < 1e-12 and abs(hmax / r.hmax - 1) < 1e-12
    assert emax > 0.9 * nz and 0 < 100 * hmax < emax
    assert np.argmax(r.emax_hist) != np.argmax(r.hmax_hist)              # the two maxima are reached at different steps


# ------------------------------------------------------------------------------------------------
# R4  CPML sample POSITIONS (integer E positions, half-integer H positions, low and high face)
# ------------------------------------------------------------------------------------------------
def _read_cpml_golden(golden_dir):
    rows = {}
    for line in open(os.path.join(golden_dir, "cpml_profile_lo4_hi3.txt")):
        if line.startswith("#") or not line.strip():
            continue
        u, rho_e, ce, rho_h, ch = [x.strip() for x in line.split("|")]
        rows[int(u)] = (Fraction(rho_e), [float(x) for x in ce.split()], Fraction(rho_h), [float(x) for x in ch.split()])
    return rows


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_R4_cpml_profile_positions_against_hand_written_fixture(golden_dir, axis):
    """tests/golden/cpml_profile_lo4_hi3.txt lists, for n = 12, lo = 4, hi = 3, the depth rho at every E index and every
    H index (typed by hand from R4's two sentences) and b, c, 1/kappa from the closed forms.  A half-cell offset, a
    swapped E/H profile or a mirrored high side changes rho at every slab index."""
    rows = _read_cpml_golden(golden_dir)
    d = 5e-9
    dt = d / (2.0 * C0)
    n = [6, 6, 6]
    n[axis] = 12
    pml = [0] * 6
    pml[2 * axis], pml[2 * axis + 1] = 4, 3
    o = YeeOracle(n[0], n[1], n[2], d, d, d, dt)
    o.set_boundary(pml, [3.0, 1.0, 5.0, 0.05, 0.8, 4.0])
    o.commit()
    prof = o.cpml_profile(axis)
    assert sorted(rows) == [0, 1, 2, 3, 9, 10, 11]
    for u, (rho_e, ce, rho_h, ch) in rows.items():
        for name, ref in zip(("bE", "cE", "ikE"), ce):
            assert abs(prof[name][u] - ref) <= 1e-14, (name, u)
        for name, ref in zip(("bH", "cH", "ikH"), ch):
            assert abs(prof[name][u] - ref) <= 1e-14, (name, u)
    for u in range(4, 9):                                                # interior: no absorption, no stretching
        for name, ref in (("bE", 1), ("cE", 0), ("ikE", 1), ("bH", 1), ("cH", 0), ("ikH", 1)):
            assert prof[name][u] == ref
    # the other axes have no layer at all
    for a in range(3):
        if a != axis:
            q = o.cpml_profile(a)
            assert (q["cE"] == 0).all() and (q["cH"] == 0).all() and (q["ikE"] == 1).all()
    # the fixture's own depth table is monotone towards the walls and E/H interleave by half a cell
    assert [rows[u][0] for u in (0, 1, 2, 3)] == [Fraction(4 - u, 4) for u in (0, 1, 2, 3)]
    assert [rows[u][2] for u in (0, 1, 2, 3)] == [Fraction(7 - 2 * u, 8) for u in (0, 1, 2, 3)]
    assert [rows[u][0] for u in (9, 10, 11)] == [Fraction(0), Fraction(1, 3), Fraction(2, 3)]
    assert [rows[u][2] for u in (9, 10, 11)] == [Fraction(1, 6), Fraction(1, 2), Fraction(5, 6)]


# ------------------------------------------------------------------------------------------------
# P11  linearity and reciprocity
# ------------------------------------------------------------------------------------------------
def test_P11_linearity_in_source_amplitude():
    w = W.random_box(5, steps=30)
    o1 = YeeOracle.from_workload(w)
    w["ports"][0]["amp"] = -2.5
    o2 = YeeOracle.from_workload(w)
    o1.step(30); o2.step(30)
    for c in range(6):
        a, b = o1.read_field(c), o2.read_field(c)
        assert np.abs(b + 2.5 * a).max() <= 1e-12 * np.abs(b).max()


def test_P11_reciprocity_on_parallel_plate_with_obstacle():
    """S*_21 = S*_12 for a reciprocal two-port: drive from port 1 (+x) and from port 2 (-x)."""
    fr = np.linspace(5e12, 100e12, 8)
    S = {}
    for drive in (0, 1):
        res = {}
        for run in ("inc", "tot"):
            w = W.parallel_plate(nx=300, ip1=90, ip2=210, isrc=70, freqs=fr, steps=5000, sig_dt=30.0)
            if drive == 1:
                p0, p1 = w["ports"]
                src = {k: p0[k] for k in ("sj0", "sj1", "sk0", "sk1", "waveform", "amp", "t0", "sigma", "f0")}
                p1.update(src); p1["is"] = 300 - 70; p1["has_source"] = 1; p0["has_source"] = 0
            if run == "tot":
                e = [a.copy() for a in w["materials"]["eps_r"]]
                for c in range(3):
                    e[c][:, :, 140:155] = 6.0          # asymmetric dielectric slug
                    e[c][:, :, 155:160] = 2.0
                w["materials"]["eps_r"] = e
            o = YeeOracle.from_workload(w)
            o.step(5000)
            res[run] = [o.read_port_dft(p) for p in (0, 1)]
        sgn = 1.0 if drive == 0 else -1.0              # DESIGN.md R9: far-end drive reverses the loop sense
        Vi = [res["inc"][p][0] for p in (0, 1)]
        Ii = [sgn * res["inc"][p][1] for p in (0, 1)]
        Vt = [res["tot"][p][0] for p in (0, 1)]
        S[drive] = osp.s_star_column(drive, Vi, Ii, Vt)
    S21, S12 = np.array(S[0][1]), np.array(S[1][0])
    assert np.abs(S21).min() > 0.1
    assert np.abs(S21 - S12).max() < 1e-3


# ------------------------------------------------------------------------------------------------
# P9  microstrip sanity (loose): Z_r and eps_eff of C1's cross-section vs the quasi-static textbook formula
# ------------------------------------------------------------------------------------------------
def test_P9_microstrip_sanity_loose():
    fr = np.linspace(20e12, 60e12, 5)
    w = W.microstrip_c1(nx=128, steps=3000, precision=64, freqs=fr)
    w["ports"][0]["ip"], w["ports"][1]["ip"] = 40, 100     # both planes clear of the source's near field
    o = YeeOracle.from_workload(w)
    o.step(3000)
    V1, I1 = o.read_port_dft(0)
    V2, I2 = o.read_port_dft(1)
    Zr = V1 / I1
    # textbook quasi-static microstrip (Pozar [3]; the same formula family that gives the paper's 25-ohm design
    # point) for w/h = 8/12, eps_r = 3.9 -- thick strip in a tight box, hence +-20 %
    u, er = 8 / 12, 3.9
    ee = (er + 1) / 2 + (er - 1) / 2 / math.sqrt(1 + 12 / u)
    z0 = 60 / math.sqrt(ee) * math.log(8 / u + u / 4)
    assert (np.real(Zr) < 0).all()
    assert np.abs(np.abs(Zr) / z0 - 1).max() < 0.2
    L = (100 - 40) * w["dx"]
    beta = -np.unwrap(np.angle(V2 / V1)) / L
    eps_eff = (beta * C0 / (2 * np.pi * fr)) ** 2
    assert np.abs(eps_eff / ee - 1).max() < 0.2


def test_fp32_instantiation_tracks_fp64():
    """The fp32 yardstick (R14) is the same algorithm: it agrees with fp64 to fp32 rounding."""
    w = W.random_box(6, steps=50)
    a = YeeOracle.from_workload(w, track_max=True)
    b = YeeOracle.from_workload(w, f32=True)
    a.step(50); b.step(50)
    emax, hmax = a.running_max()
    for c in range(6):
        e = np.abs(a.read_field(c) - b.read_field(c)).max() / (emax if c < 3 else hmax)
        assert 0 < e < 1e-5


def test_R31_far_end_drive_orientation_and_reciprocity_of_the_protocol():
    """Driving the parallel-plate line from its far port (workloads.drive_port) sends the wave towards -x: V/I changes
    sign, and the oriented reference impedance Z_r = -d V/I (R31; d = +1 for a +x drive, -1 for a -x drive) is
    +eta0 gap/width for both drives -- the sign Eq. 5 needs.  The two S*_21 of the two-run-per-port protocol
    agree: the uniform vacuum line is reciprocal."""
    fr = np.linspace(5e12, 250e12, 24)
    w = W.parallel_plate(freqs=fr, steps=3000)
    Z_th = ETA0 * w["gap_m"] / w["width_m"]
    S21 = []
    for j in (0, 1):
        wj, d = W.drive_port(w, j)
        assert d == (1, -1)[j]
        o = YeeOracle.from_workload(wj)
        o.step(3000)
        V = [o.read_port_dft(p)[0] for p in range(2)]
        I = [o.read_port_dft(p)[1] for p in range(2)]
        zr = -d * V[j] / I[j]
        assert np.abs(zr.real / Z_th - 1).max() < 1e-3 and np.abs(zr.imag).max() < 0.1 * Z_th
        S = osp.s_star_column(j, V, I, V)
        S21.append(np.array(S[1 - j]))
    assert np.abs(S21[0] - S21[1]).max() < 1e-5
