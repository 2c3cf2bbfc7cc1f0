"""S* -> S at 50 ohm (Eq. 5-6) and the phase delay (Eq. 8) -- oracle side (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Follows PAPER.md:68-87 (Eq. 5-6) one frequency at a time, plain Python complex numbers and explicit small-matrix loops
(Gauss-Jordan inverse), no numpy:

    S = A^-1 . (S* - conj(B)) . (I - B . S*)^-1 . conj(A)                                   (Eq. 5)
    A = Gstar^-1 . G . (I - conj(B))
    B = (Zstar - Z_r) . (Zstar + conj(Z_r))^-1                                              (R29)
    G_ii = 1/sqrt(|Re Z_r(y_i)|),  Z_r,ii = Z_r(y_i),  Gstar_ii = 1/sqrt(50),  Zstar_ii = 50  (Eq. 6)

Readings (R29 = SURVEY G5): the printed B, "(Z_r* - Z_r).(Z_r* - Z_r)^-1", is the identity as it stands; the paper
cites Reveyrand's power-wave renormalisation, whose reflection term is (Z_new - Z_old)/(Z_new + conj(Z_old)).  A star on A
and B means complex conjugate, a star on Z_r and G means "the 50-ohm quantity" (the paper uses one symbol for both).
Pins (tests/test_sparam_post.py): Z_r = 50 leaves S* unchanged; a one-port load Z_L seen from a complex Z_r gives
(Z_L - 50)/(Z_L + 50); a matched line of impedance 25 ohm gives Eq. 7 with Gamma = -1/3 (with the
numerator of S21 read as (1 - Gamma^2) kappa, R30).

Phase delay (Eq. 8): tau = theta / (360 f), theta = phase of S*_ij in degrees, "unwrapped with a period
of 2 pi" along the frequency axis.
"""
import cmath
import math


def _inv(M):
    """Inverse of a small complex matrix by Gauss-Jordan elimination with partial pivoting."""
    n = len(M)
    a = [[complex(M[i][j]) for j in range(n)] + [1 + 0j if i == j else 0j for j in range(n)] for i in range(n)]
    for c in range(n):
        piv = max(range(c, n), key=lambda r: abs(a[r][c]))
        if abs(a[piv][c]) == 0.0:
            raise ZeroDivisionError("singular matrix")
        a[c], a[piv] = a[piv], a[c]
        d = a[c][c]
        a[c] = [v / d for v in a[c]]
        for r in range(n):
            if r != c and a[r][c] != 0:
                f = a[r][c]
                a[r] = [vr - f * vc for vr, vc in zip(a[r], a[c])]
    return [row[n:] for row in a]


def _mul(X, Y):
    n, m, k = len(X), len(Y[0]), len(Y)
    return [[sum(X[i][q] * Y[q][j] for q in range(k)) for j in range(m)] for i in range(n)]


def renormalize_one(S_star, Z_r, z_new=50.0):
    """Eq. 5-6 at one frequency.  S_star: N x N nested list, Z_r: N reference impedances.  Returns S (N x N)."""
    n = len(Z_r)
    I = [[1 + 0j if i == j else 0j for j in range(n)] for i in range(n)]
    B = [[(z_new - Z_r[i]) / (z_new + Z_r[i].conjugate()) if i == j else 0j for j in range(n)] for i in range(n)]
    Bc = [[B[i][j].conjugate() for j in range(n)] for i in range(n)]
    G = [1.0 / math.sqrt(abs(Z_r[i].real)) for i in range(n)]
    Gs = 1.0 / math.sqrt(z_new)
    A = [[(1.0 / Gs) * G[i] * (I[i][j] - Bc[i][j]) for j in range(n)] for i in range(n)]
    Ac = [[A[i][j].conjugate() for j in range(n)] for i in range(n)]
    Ss = [[complex(S_star[i][j]) for j in range(n)] for i in range(n)]
    left = _mul(_inv(A), [[Ss[i][j] - Bc[i][j] for j in range(n)] for i in range(n)])
    BS = _mul(B, Ss)
    mid = _inv([[I[i][j] - BS[i][j] for j in range(n)] for i in range(n)])
    return _mul(_mul(left, mid), Ac)


def renormalize(S_star, Z_r, z_new=50.0):
    """S_star[i][j][m], Z_r[i][m] over frequencies m -> S[i][j][m]."""
    n = len(Z_r)
    nf = len(Z_r[0])
    out = [[[0j] * nf for _ in range(n)] for _ in range(n)]
    for m in range(nf):
        S = renormalize_one([[S_star[i][j][m] for j in range(n)] for i in range(n)], [complex(Z_r[i][m]) for i in range(n)], z_new)
        for i in range(n):
            for j in range(n):
                out[i][j][m] = S[i][j]
    return out


def unwrapped_phase_deg(s):
    """Phase of the complex sequence s in degrees, unwrapped with a period of 2 pi (jumps larger than pi removed)."""
    th = []
    off = 0.0
    prev = None
    for v in s:
        p = cmath.phase(v)
        if prev is not None:
            d = p - prev
            if d > math.pi:
                off -= 2 * math.pi
            elif d < -math.pi:
                off += 2 * math.pi
        prev = p
        th.append(math.degrees(p + off))
    return th


def phase_delay(s, freqs):
    """Eq. 8: tau_m = theta_m / (360 f_m)."""
    return [t / (360.0 * f) for t, f in zip(unwrapped_phase_deg(s), freqs)]
