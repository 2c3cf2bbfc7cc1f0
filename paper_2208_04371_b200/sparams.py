"""S* from the port DFTs of an "inc" and a "tot" run (host side of the path; Eq. 1-2).

  Z_r(y_p, f) = F[V_inc(y_p)] / F[I_inc(y_p)]                                   (Eq. 2)
  S*_jj       = (F[V_tot(y_j)] - F[V_inc(y_j)]) / F[V_inc(y_j)]                 (Eq. 1, i = j)
  S*_ij       = F[V_tot(y_i)] / F[V_inc(y_j)] * sqrt(Z_r(y_j) / Z_r(y_i))       (Eq. 1, i != j; principal root)
O(ports * freqs) complex operations on the numbers fdtd_read_port_dft returns.
"""
import numpy as np


def reference_impedance(V_inc, I_inc):
    return np.asarray(V_inc, dtype=np.complex128) / np.asarray(I_inc, dtype=np.complex128)


def s_star_column(j, V_inc, I_inc, V_tot):
    """Column j of S* (port j drives).  Inputs: arrays [ports, freqs].  Returns S[ports, freqs]."""
    V_inc = np.asarray(V_inc, dtype=np.complex128)
    V_tot = np.asarray(V_tot, dtype=np.complex128)
    zr = reference_impedance(V_inc, I_inc)
    S = V_tot / V_inc[j][None, :] * np.sqrt(zr[j][None, :] / zr)
    S[j] = (V_tot[j] - V_inc[j]) / V_inc[j]
    return S


def renormalize(S_star, Z_r, z_new=50.0):
    """S* (power waves on the per-port reference impedances Z_r) -> S on z_new ohm at every port (Eq. 5-6,
    PAPER.md:68-87, after Reveyrand; readings R29 in DESIGN.md).  S_star: [N, N, F], Z_r: [N, F] with Re Z_r > 0
    (orient the current along the incident wave).  Returns [N, N, F].

        B = (z_new - Z_r) / (z_new + conj Z_r)          (diagonal; the printed form is the identity, R29)
        A = sqrt(z_new) / sqrt|Re Z_r| * (1 - conj B)   (diagonal, Eq. 6: G = 1/sqrt|Re Z_r|, G* = 1/sqrt(z_new))
        S = A^-1 (S* - conj B) (I - B S*)^-1 conj A
    Solved per frequency with one batched linear solve instead of explicit inverses.
    """
    S = np.moveaxis(np.asarray(S_star, dtype=np.complex128), 2, 0)          # [F, N, N]
    Z = np.asarray(Z_r, dtype=np.complex128).T                              # [F, N]
    n = Z.shape[1]
    b = (z_new - Z) / (z_new + np.conj(Z))
    a = np.sqrt(z_new) / np.sqrt(np.abs(Z.real)) * (1.0 - np.conj(b))
    eye = np.eye(n)[None]
    num = S - np.conj(b)[:, :, None] * eye                                   # S* - conj B
    den = eye - b[:, :, None] * S                                            # I - B S*
    # X = num den^-1  <=>  den^T X^T = num^T
    X = np.swapaxes(np.linalg.solve(np.swapaxes(den, 1, 2), np.swapaxes(num, 1, 2)), 1, 2)
    out = X * np.conj(a)[:, None, :] / a[:, :, None]                         # A^-1 X conj A
    return np.moveaxis(out, 0, 2)


def phase_delay(s, freqs):
    """Eq. 8: tau = theta / (360 f), theta = phase of S*_ij in degrees unwrapped along frequency.
    With this library's DFT kernel e^{-j 2 pi f t} a delayed signal has a falling phase, so tau is negative for a
    physical delay; the paper's sign is that of its own time convention (R30)."""
    th = np.degrees(np.unwrap(np.angle(np.asarray(s, dtype=np.complex128))))
    return th / (360.0 * np.asarray(freqs, dtype=np.float64))


def abcd_from_s(S, z0=50.0):
    """Two-port S (on the real reference z0 at both ports, [2, 2, F]) -> ABCD chain matrix [2, 2, F]
    ("S* can also be converted to an ABCD matrix"; the standard two-port conversion, Pozar [3])."""
    S = np.asarray(S, dtype=np.complex128)
    s11, s12, s21, s22 = S[0, 0], S[0, 1], S[1, 0], S[1, 1]
    A = ((1 + s11) * (1 - s22) + s12 * s21) / (2 * s21)
    B = z0 * ((1 + s11) * (1 + s22) - s12 * s21) / (2 * s21)
    Cc = ((1 - s11) * (1 - s22) - s12 * s21) / (2 * s21) / z0
    D = ((1 - s11) * (1 + s22) + s12 * s21) / (2 * s21)
    return np.array([[A, B], [Cc, D]])


def telegrapher_from_abcd(abcd, length, freqs):
    """Overall characteristic impedance and per-unit-length R, L, G, C of the "simplest Telegrapher's model" (PAPER.md:89,
    128-134): a uniform line of the given length with the same ABCD matrix, A = cosh(gamma l), B = Z0 sinh(gamma l),
    C = sinh(gamma l) / Z0:  Z0 = sqrt(B / C), gamma = acosh(A) / l (branch unwrapped along frequency, Re gamma >= 0),
    R + j w L = gamma Z0,  G + j w C = gamma / Z0.  Returns a dict of arrays over frequency."""
    A, Bm, Cm = abcd[0, 0], abcd[0, 1], abcd[1, 0]
    f = np.asarray(freqs, dtype=np.float64)
    z0 = np.sqrt(Bm / Cm)
    z0 = np.where(z0.real < 0, -z0, z0)
    gl = np.arccosh(A)                                   # principal value: Re >= 0, Im in [0, pi] (beta l folded)
    gl = np.where(gl.real < 0, -gl, gl)
    # unfold beta l: sinh(gamma l) = B / Z0 decides the sign of the imaginary part, then unwrap along frequency
    sh = Bm / z0
    im = np.where(np.sign(np.sinh(gl).imag) == np.sign(sh.imag), gl.imag, -gl.imag)
    beta_l = np.unwrap(im)
    gamma = (gl.real + 1j * beta_l) / length
    w = 2 * np.pi * f
    series, shunt = gamma * z0, gamma / z0
    return {"Z0": z0, "gamma": gamma, "R": series.real, "L": series.imag / w, "G": shunt.real, "C": shunt.imag / w}
