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
