"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic: it only produces *inputs* -- grid sizes, dt, the
material maps (component-sampled eps_r / sigma / mu_r, either as a uint8 index into a small table or as
full arrays), CPML thickness and constants, port boxes and loops, DFT frequency lists, step counts.
It imports neither oracle/ nor paper_2208_04371_b200/.

The five configurations C0..C4 are the strings of BASELINE.json:configs made concrete (recipe in
DESIGN.md "Input recipe").  No public dataset stands behind them: the paper's own
geometries (PAPER.md:91-95 microstrip, PAPER.md:112-116 CMOS line) give the *shape* (nanometre cells,
attosecond steps, layered dielectric + long conductors + a discontinuity, PML on every face but a PEC
ground, two-run inc/tot protocol).  All random draws: numpy.random.Generator(PCG64(seed)), seed =
2208 + config index, in the order written here.

A workload is a plain dict:
  nx ny nz dx dy dz dt precision(32|64) pml[6] cpml[6]|None steps
  materials: {"mode": "indexed", "idx": uint8[nz,ny,nx], "eps_r": [ne,3], "sigma": [ne,3], "mu_r": None|[ne,3]}
           | {"mode": "full", "eps_r": [3 x float64[nz,ny,nx]], "sigma": [3 x ...], "mu_r": None|[3 x ...]}
  ports: list of dicts with the fields of fdtd_port (include/fdtd.h)
  freqs: float64[nf]
Arrays are indexed [k, j, i] (x fastest in memory), component-sampled: cell (i,j,k) owns
Ex(i+1/2,j,k), Ey(i,j+1/2,k), Ez(i,j,k+1/2), Hx(i,j+1/2,k+1/2), Hy(i+1/2,j,k+1/2), Hz(i+1/2,j+1/2,k).
"""
from __future__ import annotations

import math

import numpy as np

C0_LIGHT = 299792458.0
W_DGAUSS, W_GAUSS, W_GSINE = 0, 1, 2
INF = float("inf")
SIGMA_CU = 5.8e7


def cfl_limit(dx, dy, dz):
    """Largest stable dt on the grid (an *input* value; PAPER.md:93, 116 quote 0.9 of it)."""
    return 1.0 / (C0_LIGHT * math.sqrt(1.0 / dx**2 + 1.0 / dy**2 + 1.0 / dz**2))


def rng_for(seed):
    return np.random.Generator(np.random.PCG64(seed))


def band(nf, f_lo=1e9, f_hi=500e9):
    return np.linspace(f_lo, f_hi, nf)


# --------------------------------------------------------------------------------------------------
# Voxeliser: paints palette ids per E component, then compresses to (idx, table).
# --------------------------------------------------------------------------------------------------
class Painter:
    """Component-sampled material painter (R12 = SURVEY G12).

    A dielectric layer between planes k0 and k1 gives Ex, Ey on planes k0 < k < k1 and Ez(k+1/2),
    k0 <= k < k1, the layer's eps; the interface plane between two layers gets the mean eps for Ex, Ey.
    A conductor occupying node box [i0..i1]x[j0..j1]x[k0..k1] claims every edge on its closed surface
    and in its interior.
    """

    def __init__(self, nx, ny, nz):
        self.shape = (nz, ny, nx)
        self.pal = [(1.0, 0.0)]  # palette id 0 = vacuum (eps_r, sigma)
        self.m = [np.zeros(self.shape, dtype=np.uint8) for _ in range(3)]

    def pid(self, eps_r, sigma=0.0):
        key = (float(eps_r), float(sigma))
        if key not in self.pal:
            self.pal.append(key)
            assert len(self.pal) <= 256
        return self.pal.index(key)

    def layers(self, bounds, eps_list):
        """bounds: k0 < k1 < ... (len = len(eps_list)+1), layer l spans planes bounds[l]..bounds[l+1]."""
        nz = self.shape[0]
        for l, er in enumerate(eps_list):
            k0, k1 = bounds[l], min(bounds[l + 1], nz)
            p = self.pid(er)
            self.m[2][k0:k1] = p                      # Ez(k+1/2), k0 <= k < k1
            self.m[0][k0 + 1:k1] = p                  # Ex, Ey strictly inside
            self.m[1][k0 + 1:k1] = p
            lower = eps_list[l - 1] if l > 0 else er  # plane k0: mean with the layer below
            pm = self.pid(0.5 * (lower + er))
            if k0 < nz:
                self.m[0][k0] = pm
                self.m[1][k0] = pm

    def conductor(self, i0, i1, j0, j1, k0, k1, sigma=INF, eps_r=1.0):
        """Node box, all bounds inclusive."""
        nz, ny, nx = self.shape
        p = self.pid(eps_r, sigma)
        c = lambda a, n: max(0, min(a, n))
        self.m[0][c(k0, nz):c(k1 + 1, nz), c(j0, ny):c(j1 + 1, ny), c(i0, nx):c(i1, nx)] = p
        self.m[1][c(k0, nz):c(k1 + 1, nz), c(j0, ny):c(j1, ny), c(i0, nx):c(i1 + 1, nx)] = p
        self.m[2][c(k0, nz):c(k1, nz), c(j0, ny):c(j1 + 1, ny), c(i0, nx):c(i1 + 1, nx)] = p

    def indexed(self):
        P = len(self.pal)
        code = self.m[0].astype(np.uint32) + P * (self.m[1].astype(np.uint32) + P * self.m[2].astype(np.uint32))
        codes, inv = np.unique(code.reshape(-1), return_inverse=True)
        assert codes.size <= 256, "more than 256 distinct (x,y,z) material triples"
        pal = np.array(self.pal)
        trip = np.stack([codes % P, (codes // P) % P, codes // (P * P)], axis=1)
        eps = pal[trip, 0]
        sig = pal[trip, 1]
        return {"mode": "indexed", "idx": inv.astype(np.uint8).reshape(self.shape), "eps_r": eps,
                "sigma": sig, "mu_r": None}

    def full(self, eps_override=None):
        pal = np.array(self.pal)
        eps = [pal[self.m[c], 0] for c in range(3)]
        sig = [pal[self.m[c], 1] for c in range(3)]
        return {"mode": "full", "eps_r": eps, "sigma": sig, "mu_r": None}


def _port(ip, vj0, vj1, vk0, vk1, lj0, lj1, lk0, lk1, source=None):
    p = dict(has_source=0, ip=ip, vj0=vj0, vj1=vj1, vk0=vk0, vk1=vk1, lj0=lj0, lj1=lj1, lk0=lk0, lk1=lk1)
    p.update({"is": 0, "sj0": 0, "sj1": 0, "sk0": 0, "sk1": 1, "waveform": W_GAUSS, "amp": 0.0, "t0": 0.0,
              "sigma": 1.0, "f0": 0.0})
    if source:
        p.update(source)
        p["has_source"] = 1
    return p


# --------------------------------------------------------------------------------------------------
# C0  PEC cavity 32^3, fp64, one GSINE point source, 2000 steps, no PML
# --------------------------------------------------------------------------------------------------
def cavity_c0(seed=2208, n=32, steps=2000):
    d = 5e-9
    dt = 0.99 * cfl_limit(d, d, d)
    r = rng_for(seed)
    i, j, k = (int(v) for v in r.integers(4, n - 4, size=3))
    sig = 12 * dt  # DESIGN.md R15: envelope wide enough in frequency to reach the cavity modes
    src = {"is": i, "sj0": j, "sj1": j, "sk0": k, "sk1": k + 1, "waveform": W_GSINE, "amp": 1.0,
           "t0": 3 * sig, "sigma": sig, "f0": 100e9}
    # the probe fields of the source "port" are dummies placed away from the walls
    p = _port(ip=n // 2, vj0=n // 2, vj1=n // 2, vk0=1, vk1=2, lj0=n // 2, lj1=n // 2, lk0=n // 2, lk1=n // 2,
              source=src)
    one = np.ones((n, n, n))
    mats = {"mode": "full", "eps_r": [one, one, one], "sigma": [0 * one] * 3, "mu_r": None}
    return dict(name="c0", nx=n, ny=n, nz=n, dx=d, dy=d, dz=d, dt=dt, precision=64, pml=[0] * 6, cpml=None,
                materials=mats, ports=[p], freqs=np.zeros(0), steps=steps, source_cell=(i, j, k))


# --------------------------------------------------------------------------------------------------
# C1  microstrip 192x64x48, fp32, indexed
# --------------------------------------------------------------------------------------------------
def microstrip_c1(seed=2209, nx=192, steps=40000, precision=32, waveform=W_GAUSS, freqs=None):
    ny, nz, d = 64, 48, 5e-9
    dt = 0.99 * cfl_limit(d, d, d)
    pt = Painter(nx, ny, nz)
    pt.layers([0, 12, nz], [3.9, 1.0])
    pt.conductor(0, nx, 28, 36, 12, 14)                 # PEC strip 8 cells wide x 2 thick, full length
    sig = 64 * dt
    src = {"is": 20, "sj0": 28, "sj1": 36, "sk0": 0, "sk1": 12, "waveform": waveform, "amp": 1.0,
           "t0": 3 * sig, "sigma": sig, "f0": 0.0}
    box = dict(vj0=28, vj1=36, vk0=0, vk1=12, lj0=27, lj1=37, lk0=11, lk1=15)
    ports = [_port(ip=20, source=src, **box), _port(ip=nx - 20, **box)]
    return dict(name="c1", nx=nx, ny=ny, nz=nz, dx=d, dy=d, dz=d, dt=dt, precision=precision,
                pml=[8, 8, 8, 8, 0, 8], cpml=[3.0, 1.0, 1.0, 0.0, 0.8, 2.45], materials=pt.indexed(),
                ports=ports, freqs=band(128) if freqs is None else np.asarray(freqs, dtype=np.float64),
                steps=steps)


# --------------------------------------------------------------------------------------------------
# X1  the paper's microstrip verification case at paper size
# --------------------------------------------------------------------------------------------------
def microstrip_x1(nx=1000, steps=60000, precision=32, nf=79, f_hi=40e9, npml=10):
    """Z0 = 25 ohm microstrip: eps_r = 3.8, h = 1 mm = 10 cells, w/h = 5.7 (57 cells), length 100 h = 1000 cells,
    200 x 1000 x 50 cells of 0.1 mm (the paper's propagation axis y is x here), CFL number 0.9 (dt = 0.173 ps),
    differentiated-Gaussian pulse sigma = 11.254 ps, t0 = 3 sigma (Eq. 3), 60 000 steps.  Not in the paper: the PML depth
    (10 cells), the port planes (100 cells from either end), the strip thickness (a PEC sheet), the DFT band."""
    ny, nz, d = 200, 50, 1e-4
    dt = 0.9 * cfl_limit(d, d, d)
    pt = Painter(nx, ny, nz)
    pt.layers([0, 10, nz], [3.8, 1.0])
    j0, j1 = 72, 129                                     # 57 cells wide, centred
    pt.conductor(0, nx, j0, j1, 10, 10)                  # zero-thickness PEC sheet on the plane k = 10
    sig = 11.254e-12
    src = {"is": 60, "sj0": j0, "sj1": j1, "sk0": 0, "sk1": 10, "waveform": W_DGAUSS, "amp": 1.0,
           "t0": 3 * sig, "sigma": sig, "f0": 0.0}
    box = dict(vj0=j0, vj1=j1, vk0=0, vk1=10, lj0=j0 - 1, lj1=j1 + 1, lk0=9, lk1=11)
    ports = [_port(ip=100, source=src, **box), _port(ip=nx - 100, **box)]
    return dict(name="x1", nx=nx, ny=ny, nz=nz, dx=d, dy=d, dz=d, dt=dt, precision=precision,
                pml=[npml, npml, npml, npml, 0, npml], cpml=[3.0, 1.0, 1.0, 0.0, 0.8, 2.4], materials=pt.indexed(),
                ports=ports, freqs=np.linspace(f_hi / (nf + 1), f_hi, nf), steps=steps,
                theory=dict(z0=25.0, eps_r=3.8, w_over_h=5.7, gamma=-0.333))


# --------------------------------------------------------------------------------------------------
# X3-shaped  grid and time scales of the paper's CMOS transmission line
# --------------------------------------------------------------------------------------------------
def cmos_line_x3(run="tot", steps=1400000, precision=32, nf=128, npml=10):
    """200 x 120 x 800 cells of (20, 50, 5) nm = 4 x 6 x 4 um, CFL number 0.9 (dt = 0.0145 fs), Eq. 3 pulse with
    sigma = 10.146 fs, 1.4 M steps in the paper; DFT over the band the paper calls resolved, 50 GHz - 95 THz.
    The SHAPE of that workload only: Fig. 3 and the metal conductivities are not in the paper's text, so the
    cross-section below (oxide, a 30 nm thick conducting strip, a block on it in the tot run) is a stand-in."""
    nx, ny, nz = 200, 120, 800
    dx, dy, dz = 20e-9, 50e-9, 5e-9
    dt = 0.9 * cfl_limit(dx, dy, dz)
    pt = Painter(nx, ny, nz)
    pt.layers([0, 400, nz], [3.9, 1.0])
    j0, j1, k0, k1 = 40, 80, 400, 406                   # 2 um wide, 30 nm thick
    pt.conductor(0, nx, j0, j1, k0, k1, sigma=SIGMA_CU)
    if run == "tot":
        pt.conductor(90, 110, j0, j1, k1, k1 + 40, sigma=SIGMA_CU)
    sig = 10.146e-15
    src = {"is": 20, "sj0": j0, "sj1": j1, "sk0": 0, "sk1": k0, "waveform": W_DGAUSS, "amp": 1.0,
           "t0": 3 * sig, "sigma": sig, "f0": 0.0}
    box = dict(vj0=j0, vj1=j1, vk0=0, vk1=k0, lj0=j0 - 1, lj1=j1 + 1, lk0=k0 - 1, lk1=k1 + 1)
    ports = [_port(ip=30, source=src, **box), _port(ip=nx - 30, **box)]
    return dict(name="x3", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, dt=dt, precision=precision,
                pml=[npml, npml, npml, npml, 0, npml], cpml=[3.0, 1.0, 1.0, 0.0, 0.8, 2.45], materials=pt.indexed(),
                ports=ports, freqs=np.linspace(50e9, 95e12, nf), steps=steps, run=run)


# --------------------------------------------------------------------------------------------------
# C2 / C4  CMOS-like multilayer interconnect (C4 = C2 with every extent x2, fp64, full uniaxial arrays)
# --------------------------------------------------------------------------------------------------
def _interconnect(seed, mult, div, run, full, precision, npml, nf, sig_dt, nports, steps):
    """mult/div scale every extent of the 512x256x128 geometry (C2: 1/1, C4: 2/1, quarter-scale tests: 1/4)."""
    s = lambda v: (v * mult) // div
    nx, ny, nz = s(512), s(256), s(128)
    dx = dy = 2.5e-9
    dz = 5e-9
    dt = 0.99 * cfl_limit(dx, dy, dz)
    r = rng_for(seed)
    eps_layers = r.uniform(2.5, 7.5, size=6)
    eps_zz = r.uniform(2.5, 7.5, size=6) if full else eps_layers
    bounds = [s(b) for b in (0, 20, 40, 60, 80, 100)] + [nz]
    pt = Painter(nx, ny, nz)
    pt.layers(bounds, list(eps_layers))
    ja0, ja1, jb0, jb1, k0, k1 = s(108), s(118), s(138), s(148), s(44), s(48)
    k1 = max(k1, k0 + 1)
    pt.conductor(0, nx, ja0, ja1, k0, k1, sigma=SIGMA_CU)
    pt.conductor(0, nx, jb0, jb1, k0, k1, sigma=SIGMA_CU)
    if run == "tot":
        pt.conductor(s(251), s(261), ja0, ja1, s(24), k0, sigma=SIGMA_CU)     # via stub on line A
    if full:
        mats = pt.full()
        # uniaxial layers: eps_zz drawn separately; repaint Ez of the dielectric (sigma == 0) samples
        ezz = mats["eps_r"][2]
        diel = mats["sigma"][2] == 0.0
        for l in range(6):
            sl = slice(bounds[l], bounds[l + 1])
            ezz[sl] = np.where(diel[sl], eps_zz[l], ezz[sl])
    else:
        mats = pt.indexed()
    sg = sig_dt * dt
    pa, pb = s(40), nx - s(40)
    isrc = s(30)
    boxA = dict(vj0=ja0, vj1=ja1, vk0=0, vk1=k0, lj0=ja0 - 1, lj1=ja1 + 1, lk0=k0 - 1, lk1=k1 + 1)
    boxB = dict(vj0=jb0, vj1=jb1, vk0=0, vk1=k0, lj0=jb0 - 1, lj1=jb1 + 1, lk0=k0 - 1, lk1=k1 + 1)
    src = {"is": isrc, "sj0": ja0, "sj1": ja1, "sk0": 0, "sk1": k0, "waveform": W_GAUSS, "amp": 1.0,
           "t0": 3 * sg, "sigma": sg, "f0": 0.0}
    ports = [_port(ip=pa, source=src, **boxA), _port(ip=pb, **boxA)]
    if nports == 4:
        ports += [_port(ip=pa, **boxB), _port(ip=pb, **boxB)]
    np_ = npml
    return dict(nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, dt=dt, precision=precision,
                pml=[np_, np_, np_, np_, 0, np_], cpml=[3.0, 1.0, 1.0, 0.0, 0.8, float(np.mean(eps_layers))],
                materials=mats, ports=ports, freqs=band(nf), steps=steps, run=run)


def interconnect_c2(seed=2210, run="tot", div=1, steps=200000, npml=10, nf=256):
    w = _interconnect(seed, 1, div, run, False, 32, npml, nf, 64, 2, steps)
    w["name"] = "c2" if div == 1 else f"c2/{div}"
    return w


def interconnect_c4(seed=2212, run="tot", div=1, steps=50000, npml=12, nf=512):
    w = _interconnect(seed, 2, div, run, True, 64, npml, nf, 128, 4, steps)
    w["name"] = "c4" if div == 1 else f"c4/{div}"
    return w


# --------------------------------------------------------------------------------------------------
# C3  throughput grid 1536x768x768, fp32 + uint8 index into a 64-entry table, six-face CPML
# --------------------------------------------------------------------------------------------------
def throughput_c3(seed=2211, shape=(1536, 768, 768), steps=2000, npml=16, nf=128, nblocks=4096, div=1, kc=None):
    """kc: plane of the two port lines (default: the middle plane nz // 2; the z-slab weak-scaling grids put it in the
    middle of the lowest slab so that no interface cuts a port)."""
    nx, ny, nz = (v // div for v in shape)
    d = 5e-9
    dt = 0.99 * cfl_limit(d, d, d)
    r = rng_for(seed)
    eps = np.ones(64)
    sig = np.zeros(64)
    eps[2:] = r.uniform(1.0, 12.0, size=62)
    sig[2:] = r.choice([0.0, 1e3, SIGMA_CU], size=62, p=[0.7, 0.2, 0.1])
    sig[1] = INF
    idx = np.empty((nz, ny, nx), dtype=np.uint8)
    k = 0
    while k < nz:                                        # random z-layers, thickness U{8..64}
        t = max(1, int(r.integers(8, 65)) // div)
        idx[k:k + t] = int(r.integers(2, 64))
        k += t
    for _ in range(max(1, nblocks // div**3)):           # random axis-aligned blocks, edge U{16..128}
        e = np.maximum(1, r.integers(16, 129, size=3) // div)
        o = [int(r.integers(0, n)) for n in (nx, ny, nz)]
        idx[o[2]:o[2] + e[2], o[1]:o[1] + e[1], o[0]:o[0] + e[0]] = int(r.integers(2, 64))
    # two PEC lines (10 x 4 cells) in a vacuum corridor (+-24 cells) along x, for the ports
    cw, ch, cor = max(2, 10 // div), max(1, 4 // div), max(3, 24 // div)
    kc = nz // 2 if kc is None else int(kc)
    lines = []
    for jc in (ny // 3, (2 * ny) // 3):
        idx[kc - cor:kc + ch + cor, jc - cor:jc + cw + cor, :] = 0
        idx[kc:kc + ch, jc:jc + cw, :] = 1
        lines.append(jc)
    sg = 64 * dt
    ports = []
    x0 = max(npml + 4, 48 // div)
    for n, jc in enumerate(lines):
        box = dict(vj0=jc, vj1=jc + cw, vk0=kc - cor, vk1=kc, lj0=jc - 1, lj1=jc + cw + 1, lk0=kc - 1,
                   lk1=kc + ch + 1)
        src = None
        if n == 0:
            src = {"is": x0, "sj0": jc, "sj1": jc + cw, "sk0": kc - cor, "sk1": kc, "waveform": W_GAUSS,
                   "amp": 1.0, "t0": 3 * sg, "sigma": sg, "f0": 0.0}
        ports.append(_port(ip=x0, source=src, **box))
        ports.append(_port(ip=nx - x0, **box))
    table_eps = np.repeat(eps[:, None], 3, axis=1)
    table_sig = np.repeat(sig[:, None], 3, axis=1)
    mats = {"mode": "indexed", "idx": idx, "eps_r": table_eps, "sigma": table_sig, "mu_r": None}
    return dict(name="c3" if div == 1 else f"c3/{div}", nx=nx, ny=ny, nz=nz, dx=d, dy=d, dz=d, dt=dt,
                precision=32, pml=[npml] * 6, cpml=[3.0, 1.0, 1.0, 0.0, 0.8, float(np.mean(eps[2:]))],
                materials=mats, ports=ports, freqs=band(nf), steps=steps)


# --------------------------------------------------------------------------------------------------
# Small cases used by the pins and the parity tests
# --------------------------------------------------------------------------------------------------
def parallel_plate(nx=240, ny=2, gap=8, d=5e-9, npml=10, steps=3000, sig_dt=24.0, waveform=W_GAUSS,
                   freqs=None, ip1=60, ip2=180, isrc=40, precision=64):
    """Vacuum parallel-plate line (oracle-only pin; needs the oracle's periodic-y option).

    PEC ground at z = 0, a zero-thickness PEC sheet on plane k = gap (Ex, Ey there are PEC), quiet
    vacuum above it up to nz = 2*gap; periodic in y; CPML on both x faces.  The TEM mode in the lower
    gap has Z = eta0 * d / w with d = gap*dz and w = (number of loop columns)*dy."""
    nz = 2 * gap
    dt = 0.99 * cfl_limit(d, d, d)
    one = np.ones((nz, ny, nx))
    sx = np.zeros((nz, ny, nx))
    sx[gap] = INF
    mats = {"mode": "full", "eps_r": [one] * 3, "sigma": [sx, sx.copy(), np.zeros((nz, ny, nx))], "mu_r": None}
    sg = sig_dt * dt
    src = {"is": isrc, "sj0": 0, "sj1": ny - 1, "sk0": 0, "sk1": gap, "waveform": waveform, "amp": 1.0,
           "t0": 3 * sg, "sigma": sg, "f0": 0.0}
    box = dict(vj0=0, vj1=ny - 1, vk0=0, vk1=gap, lj0=1, lj1=ny - 1, lk0=gap, lk1=gap)
    ports = [_port(ip=ip1, source=src, **box), _port(ip=ip2, **box)]
    return dict(name="pplate", nx=nx, ny=ny, nz=nz, dx=d, dy=d, dz=d, dt=dt, precision=precision,
                pml=[npml, npml, 0, 0, 0, 0], cpml=None, materials=mats, periodic_y=True, ports=ports,
                freqs=np.zeros(0) if freqs is None else np.asarray(freqs, dtype=np.float64), steps=steps,
                gap_m=gap * d, width_m=(ny - 1) * d, sigma_t=sg)


def random_box(seed, nx=20, ny=14, nz=12, pml=(3, 4, 2, 3, 0, 3), indexed=True, with_mu=True, precision=64,
               nf=5, steps=40, d=(5e-9, 4e-9, 6e-9), pec_frac=0.03, cpml=(3.0, 1.0, 2.0, 0.05, 0.8, 2.0)):
    """Random blocky eps/sigma/mu in a box with mixed CPML faces and one driven port + one passive port.
    Exercises every term of the update (anisotropic spacing, kappa != 1, alpha != 0, lossy cells, PEC
    cells, mu_r != 1).  Not physical; a parity / brute-force input only."""
    r = rng_for(seed)
    dx, dy, dz = d
    dt = 0.95 * cfl_limit(dx, dy, dz)
    ne = 12
    eps = r.uniform(1.0, 12.0, size=(ne, 3))
    sig = r.choice([0.0, 1e3, 2e5, SIGMA_CU], size=(ne, 3), p=[0.55, 0.2, 0.15, 0.1])
    mu = r.uniform(1.0, 2.0, size=(ne, 3)) if with_mu else None
    eps[0] = 1.0
    sig[0] = 0.0
    sig[1] = INF                                           # entry 1 = PEC
    idx = np.zeros((nz, ny, nx), dtype=np.uint8)
    for _ in range(10):
        e = r.integers(2, 8, size=3)
        o = [int(r.integers(0, n)) for n in (nx, ny, nz)]
        idx[o[2]:o[2] + e[2], o[1]:o[1] + e[1], o[0]:o[0] + e[0]] = int(r.integers(2, ne))
    pec = r.random((nz, ny, nx)) < pec_frac
    idx[pec] = 1
    # keep the port neighbourhood free of PEC so that the source is not sitting on metal
    jc, kc = ny // 2, nz // 2
    i_s, i_1, i_2 = pml[0] + 2, pml[0] + 3, nx - pml[1] - 3
    for ii in (i_s, i_1, i_2):
        blk = idx[kc - 3:kc + 3, jc - 3:jc + 3, ii]
        blk[blk == 1] = 0
    if indexed:
        mats = {"mode": "indexed", "idx": idx, "eps_r": eps, "sigma": sig, "mu_r": mu}
    else:
        mats = {"mode": "full", "eps_r": [eps[idx, c] for c in range(3)], "sigma": [sig[idx, c] for c in range(3)],
                "mu_r": None if mu is None else [mu[idx, c] for c in range(3)]}
    sg = 6 * dt
    box = dict(vj0=jc - 1, vj1=jc + 1, vk0=kc - 2, vk1=kc, lj0=jc - 1, lj1=jc + 1, lk0=kc - 1, lk1=kc + 1)
    src = {"is": i_s, "sj0": jc - 1, "sj1": jc + 1, "sk0": kc - 2, "sk1": kc, "waveform": W_DGAUSS, "amp": 1.0,
           "t0": 3 * sg, "sigma": sg, "f0": 0.0}
    ports = [_port(ip=i_1, source=src, **box), _port(ip=i_2, **box)]
    fmax = 1.0 / (math.sqrt(2.0) * math.pi * sg)
    return dict(name=f"rbox{seed}", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, dt=dt, precision=precision,
                pml=list(pml), cpml=list(cpml) if cpml is not None else None, materials=mats, ports=ports,
                freqs=np.linspace(0.2 * fmax, 2 * fmax, nf), steps=steps)


def drive_port(w, j):
    """Copy of workload w in which port j carries the (single) source instead of the port that has it now.

    The waveform is kept; the source box becomes port j's voltage box, on a plane as far outside port j (towards the nearer
    x end of the line) as the original source plane is outside its own port.  Returns (workload, direction): direction is
    +1 when the incident wave crosses port j travelling towards +x, -1 otherwise (one inc/tot pair of
    runs per driving port).  Input bookkeeping only: none of the method's arithmetic lives here."""
    ports = [dict(q) for q in w["ports"]]
    src = [q for q in ports if q["has_source"]]
    assert len(src) == 1, "drive_port expects exactly one driving port"
    s0 = src[0]
    off = abs(s0["ip"] - s0["is"])
    wave = {k: s0[k] for k in ("waveform", "amp", "t0", "sigma", "f0")}
    for q in ports:
        q.update(has_source=0, amp=0.0)
    t = ports[j]
    direction = 1 if t["ip"] < w["nx"] // 2 else -1
    t.update(wave)
    t.update({"has_source": 1, "is": t["ip"] - direction * off, "sj0": t["vj0"], "sj1": t["vj1"], "sk0": t["vk0"],
              "sk1": t["vk1"]})
    assert 0 <= t["is"] < w["nx"]
    return dict(w, ports=ports), direction


def weak_scaling_600(n_slabs=1, steps=100, edge=600):
    """The per-GPU load of the paper's weak-scaling study (Table I: 600^3 cells per GPU), stacked along z:
    edge x edge x (edge * n_slabs) cells of C3's generator (same block density, 16-cell CPML on all six faces, 4 ports on
    two lines through the lowest slab)."""
    vol = n_slabs * edge**3 / (1536 * 768 * 768)
    w = throughput_c3(shape=(edge, edge, edge * n_slabs), steps=steps, nblocks=max(1, int(4096 * vol)), kc=edge // 2)
    w["name"] = f"weak{edge}x{n_slabs}"
    return w


def get(name, **kw):
    return {"c0": cavity_c0, "c1": microstrip_c1, "c2": interconnect_c2, "c3": throughput_c3,
            "c4": interconnect_c4}[name](**kw)
