"""A second, structurally different formulation of the same time step, for tiny grids only (pin P10).

Whole-array numpy: zero-padded np.diff for the curls, psi arrays on the WHOLE grid (c = 0 outside the
slabs), complex exponentials for the DFT.  It shares nothing with oracle/yee_oracle.cpp (which loops
cell by cell with slab-compact psi) nor with the CUDA path.  A wrong index, sign, transposed operand,
slab offset or profile position in either one makes the two disagree.
"""
import numpy as np

C = 299792458.0
MU0 = 4e-7 * np.pi
EPS0 = 1.0 / (MU0 * C * C)
ETA0 = MU0 * C


def _fwd(a, axis, d):
    pad = [(0, 0)] * 3
    pad[axis] = (0, 1)
    return np.diff(np.pad(a, pad), axis=axis) / d


def _bwd(a, axis, d):
    pad = [(0, 0)] * 3
    pad[axis] = (1, 0)
    return np.diff(np.pad(a, pad), axis=axis) / d


def _g(kind, t, t0, s, f0):
    u = (t - t0) / s
    if kind == 0:
        return -2 * u * np.exp(-u * u)
    if kind == 1:
        return np.exp(-u * u)
    return np.sin(2 * np.pi * f0 * (t - t0)) * np.exp(-u * u)


class NumpyYee:
    AX = {"x": 2, "y": 1, "z": 0}  # array axis of each space axis ([k, j, i] storage)

    def __init__(self, w):
        self.w = w
        nx, ny, nz = w["nx"], w["ny"], w["nz"]
        self.sh = (nz, ny, nx)
        self.d = {"x": w["dx"], "y": w["dy"], "z": w["dz"]}
        self.n = {"x": nx, "y": ny, "z": nz}
        self.dt = dt = w["dt"]
        m = w["materials"]
        if m["mode"] == "indexed":
            idx = np.asarray(m["idx"])
            eps = [np.asarray(m["eps_r"])[idx, c] for c in range(3)]
            sig = [np.asarray(m["sigma"])[idx, c] for c in range(3)]
            mu = [np.ones(self.sh)] * 3 if m.get("mu_r") is None else [np.asarray(m["mu_r"])[idx, c] for c in range(3)]
        else:
            eps = [np.asarray(a, dtype=float).reshape(self.sh) for a in m["eps_r"]]
            sig = [np.asarray(a, dtype=float).reshape(self.sh) for a in m["sigma"]]
            mu = [np.ones(self.sh)] * 3 if m.get("mu_r") is None else [np.asarray(a, dtype=float).reshape(self.sh) for a in m["mu_r"]]
        self.Ca, self.Cb, self.Db = [], [], []
        for c in range(3):
            with np.errstate(invalid="ignore", over="ignore"):
                a = sig[c] * dt / (2 * EPS0 * eps[c])
                ca = np.where(np.isinf(sig[c]), 0.0, (1 - a) / (1 + a))
                cb = np.where(np.isinf(sig[c]), 0.0, dt / (EPS0 * eps[c]) / (1 + a))
            self.Ca.append(ca)
            self.Cb.append(cb)
            self.Db.append(dt / (MU0 * mu[c]))
        cp = w.get("cpml") or [3.0, 1.0, 1.0, 0.0, 0.8, 1.0]
        mm, ma, kmax, amax, sfac, erp = cp
        self.prof = {}
        for ai, a in enumerate("xyz"):
            n, lo, hi = self.n[a], w["pml"][2 * ai], w["pml"][2 * ai + 1]
            smax = sfac * (mm + 1) / (ETA0 * self.d[a] * np.sqrt(erp))
            # depth into the layer from PHYSICAL coordinates: the inner CPML surfaces are the planes x = lo*d and
            # x = (n-hi)*d; an E sample sits at x = u*d, an H sample at x = (u+1/2)*d; rho = distance beyond the
            # surface / layer thickness (deliberately not the index rule the oracle and the library use)
            for tag, x in (("E", np.arange(n) * self.d[a]), ("H", (np.arange(n) + 0.5) * self.d[a])):
                x_lo, x_hi = lo * self.d[a], (n - hi) * self.d[a]
                rho = np.zeros(n)
                if lo:
                    rho = np.maximum(rho, (x_lo - x) / (lo * self.d[a]))
                if hi:
                    rho = np.maximum(rho, (x - x_hi) / (hi * self.d[a]))
                rho = np.clip(rho, 0.0, None)
                inslab = (np.arange(n) < lo) | (np.arange(n) >= n - hi)
                sg = smax * rho**mm
                kp = 1 + (kmax - 1) * rho**mm
                al = amax * (1 - rho) ** ma
                b = np.exp(-(sg / kp + al) * dt / EPS0)
                with np.errstate(invalid="ignore", divide="ignore"):
                    c = np.where(sg > 0, sg * (b - 1) / (kp * (sg + kp * al)), 0.0)
                b = np.where(inslab, b, 0.0)
                c = np.where(inslab, c, 0.0)
                ik = np.where(inslab, 1 / kp, 1.0)
                shape = [1, 1, 1]
                shape[self.AX[a]] = n
                self.prof[(a, tag)] = tuple(v.reshape(shape) for v in (b, c, ik))
        z = lambda: np.zeros(self.sh)
        self.E = {"x": z(), "y": z(), "z": z()}
        self.H = {"x": z(), "y": z(), "z": z()}
        self.psiH = {k: z() for k in ("xy", "xz", "yz", "yx", "zx", "zy")}
        self.psiE = {k: z() for k in ("xy", "xz", "yz", "yx", "zx", "zy")}
        self.nstep = 0
        self.freqs = np.asarray(w.get("freqs", []), dtype=float)
        self.Vhat = np.zeros((len(w["ports"]), self.freqs.size), dtype=complex)
        self.Ihat = np.zeros_like(self.Vhat)
        # R13: running maxima over space AND time, kept as two separate scalars, plus the per-step history
        self.emax = 0.0
        self.hmax = 0.0
        self.emax_hist, self.hmax_hist = [], []

    def _curl_term(self, psi, key, field, diff, tag):
        """derivative of `field` along axis key[1], CPML-stretched; updates psi[key] in place."""
        a = key[1]
        b, c, ik = self.prof[(a, tag)]
        der = diff(field, self.AX[a], self.d[a])
        psi[key] = b * psi[key] + c * der
        return der * ik + psi[key]

    def step(self, n=1):
        for _ in range(n):
            E, H, w = self.E, self.H, self.w
            t = lambda key, f: self._curl_term(self.psiH, key, f, _fwd, "H")
            H["x"] = H["x"] - self.Db[0] * (t("xy", E["z"]) - t("xz", E["y"]))
            H["y"] = H["y"] - self.Db[1] * (t("yz", E["x"]) - t("yx", E["z"]))
            H["z"] = H["z"] - self.Db[2] * (t("zx", E["y"]) - t("zy", E["x"]))
            t = lambda key, f: self._curl_term(self.psiE, key, f, _bwd, "E")
            ex = self.Ca[0] * E["x"] + self.Cb[0] * (t("xy", H["z"]) - t("xz", H["y"]))
            ey = self.Ca[1] * E["y"] + self.Cb[1] * (t("yz", H["x"]) - t("yx", H["z"]))
            ez = self.Ca[2] * E["z"] + self.Cb[2] * (t("zx", H["y"]) - t("zy", H["x"]))
            ex[0, :, :] = 0; ex[:, 0, :] = 0
            ey[0, :, :] = 0; ey[:, :, 0] = 0
            ez[:, 0, :] = 0; ez[:, :, 0] = 0
            E["x"], E["y"], E["z"] = ex, ey, ez
            tE, tH = (self.nstep + 1) * self.dt, (self.nstep + 0.5) * self.dt
            for p in w["ports"]:
                if p["has_source"]:
                    g = p["amp"] * _g(p["waveform"], tE, p["t0"], p["sigma"], p["f0"])
                    E["z"][p["sk0"]:p["sk1"], p["sj0"]:p["sj1"] + 1, p["is"]] += g
            for q, p in enumerate(w["ports"]):
                V = w["dz"] * E["z"][p["vk0"]:p["vk1"], p["vj0"]:p["vj1"] + 1, p["ip"]].sum() / (p["vj1"] - p["vj0"] + 1)
                hz, hy = H["z"][:, :, p["ip"]], H["y"][:, :, p["ip"]]
                I = w["dz"] * (hz[p["lk0"]:p["lk1"] + 1, p["lj1"]] - hz[p["lk0"]:p["lk1"] + 1, p["lj0"] - 1]).sum() \
                    - w["dy"] * (hy[p["lk1"], p["lj0"]:p["lj1"] + 1] - hy[p["lk0"] - 1, p["lj0"]:p["lj1"] + 1]).sum()
                self.Vhat[q] += V * np.exp(-2j * np.pi * self.freqs * tE) * self.dt
                self.Ihat[q] += I * np.exp(-2j * np.pi * self.freqs * tH) * self.dt
                self.lastV, self.lastI = V, I
            e_now = max(float(np.abs(E[c]).max()) for c in "xyz")     # E^{n+1} with the source added
            h_now = max(float(np.abs(H[c]).max()) for c in "xyz")     # H^{n+1/2}
            self.emax_hist.append(e_now)
            self.hmax_hist.append(h_now)
            self.emax, self.hmax = max(self.emax, e_now), max(self.hmax, h_now)
            self.nstep += 1

    def field(self, comp):
        return (self.E if comp < 3 else self.H)["xyz"[comp % 3]]
