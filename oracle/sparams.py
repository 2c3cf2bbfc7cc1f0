"""S* from port DFTs -- oracle side (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Follows PAPER.md:33-46 (Eq. 1-2) literally, in fp64 complex, one frequency at a time.

  Z_r(y_p, f) = F[V_inc(y_p)] / F[I_inc(y_p)]                                  (Eq. 2)
  S*_jj       = F[V_ref(y_j)] / F[V_inc(y_j)],  F[V_ref] = F[V_tot] - F[V_inc]  (Eq. 1)
  S*_ij       = F[V_tra(y_i)] / F[V_inc(y_j)] * sqrt(Z_r(y_j) / Z_r(y_i))       (Eq. 1, i != j)

Reading (R9 = SURVEY O9): the square root is the principal one; Z_r at a non-driven port
plane i comes from the same "inc" run (the incident wave crosses every port plane of the uniform line).
"""
import cmath


def reference_impedance(V_inc, I_inc):
    return [v / i for v, i in zip(V_inc, I_inc)]


def s_star_column(j, V_inc, I_inc, V_tot):
    """Column j of S* (driving port j).

    V_inc, I_inc, V_tot: lists over ports p of sequences over frequency (complex DFTs of the
    "inc" and "tot" runs at port plane p).  Returns S[p][m] for every port p and frequency m.
    """
    nports = len(V_inc)
    nf = len(V_inc[j])
    S = [[0j] * nf for _ in range(nports)]
    for m in range(nf):
        zr_j = V_inc[j][m] / I_inc[j][m]
        for p in range(nports):
            if p == j:
                S[p][m] = (V_tot[j][m] - V_inc[j][m]) / V_inc[j][m]
            else:
                zr_p = V_inc[p][m] / I_inc[p][m]
                S[p][m] = V_tot[p][m] / V_inc[j][m] * cmath.sqrt(zr_j / zr_p)
    return S
