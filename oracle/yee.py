"""ctypes front end of the CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from paper_2208_04371_b200/.

The arithmetic lives in yee_oracle.cpp; this file only marshals arguments.  The one piece of
"method" here is the expansion of an indexed material table into component-sampled arrays
(eps[c][cell] = table_eps[idx[cell]][c]), which is a gather, not arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

EX, EY, EZ, HX, HY, HZ = range(6)
W_DGAUSS, W_GAUSS, W_GSINE = 0, 1, 2

_PORT_INT_KEYS = ("has_source", "is", "sj0", "sj1", "sk0", "sk1", "waveform", "ip",
                  "vj0", "vj1", "vk0", "vk1", "lj0", "lj1", "lk0", "lk1")
_PORT_DBL_KEYS = ("amp", "t0", "sigma", "f0")


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        L.yo_constants.argtypes = [dp]
        L.yo_cfl_dt.restype = C.c_double
        L.yo_cfl_dt.argtypes = [C.c_double] * 3
        L.yo_waveform.restype = C.c_double
        L.yo_waveform.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, C.c_double]
        L.yo_create.restype = C.c_void_p
        L.yo_create.argtypes = [C.c_int] * 3 + [C.c_double] * 4 + [C.c_int, C.c_int]
        L.yo_destroy.argtypes = [C.c_void_p]
        L.yo_set_boundary.argtypes = [C.c_void_p, C.POINTER(C.c_int), dp]
        L.yo_set_materials.argtypes = [C.c_void_p] + [dp] * 9
        L.yo_add_port.argtypes = [C.c_void_p, C.POINTER(C.c_int), dp]
        L.yo_set_dft.argtypes = [C.c_void_p, dp, C.c_int]
        L.yo_set_track_max.argtypes = [C.c_void_p, C.c_int]
        L.yo_commit.argtypes = [C.c_void_p]
        L.yo_step.argtypes = [C.c_void_p, C.c_long]
        L.yo_step_count.restype = C.c_long
        L.yo_step_count.argtypes = [C.c_void_p]
        L.yo_read_field.argtypes = [C.c_void_p, C.c_int, dp]
        L.yo_write_field.argtypes = [C.c_void_p, C.c_int, dp]
        L.yo_read_port_dft.argtypes = [C.c_void_p, C.c_int, dp, dp]
        L.yo_read_port_last.argtypes = [C.c_void_p, C.c_int, dp, dp]
        L.yo_running_max.argtypes = [C.c_void_p, dp, dp]
        L.yo_psi_norms.argtypes = [C.c_void_p, dp]
        L.yo_cpml_profile.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def constants():
    """(c, mu0, eps0, eta0) as the oracle uses them."""
    out = np.zeros(4)
    lib().yo_constants(_dp(out))
    return tuple(out)


def cfl_dt(dx, dy, dz):
    return lib().yo_cfl_dt(dx, dy, dz)


def waveform(kind, t, t0, sigma, f0=0.0):
    L = lib()
    t = np.atleast_1d(np.asarray(t, dtype=np.float64))
    return np.array([L.yo_waveform(kind, float(x), t0, sigma, f0) for x in t])


def num_threads():
    """Threads the OpenMP loops of the oracle will use."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env.split(",")[0])
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def set_num_threads(n):
    """Number of threads the oracle's OpenMP loops use from now on (bench.py's one-thread figure): omp_set_num_threads of
    the OpenMP runtime the oracle library is linked against."""
    lib()
    C.CDLL("libgomp.so.1").omp_set_num_threads(int(n))


class YeeOracle:
    def __init__(self, nx, ny, nz, dx, dy, dz, dt, f32=False, periodic_y=False):
        self.L = lib()
        self.shape = (nx, ny, nz)
        self.N = nx * ny * nz
        self.dt = dt
        self.h = self.L.yo_create(nx, ny, nz, dx, dy, dz, dt, int(f32), int(periodic_y))
        if not self.h:
            raise ValueError("yo_create rejected the grid (n<2, d<=0, or dt above the CFL limit)")
        self.nf = 0
        self.nports = 0

    def __del__(self):
        if getattr(self, "h", None):
            self.L.yo_destroy(self.h)
            self.h = None

    # ---- setup ---------------------------------------------------------------------------------
    def set_boundary(self, pml, cpml=None):
        p = (C.c_int * 6)(*[int(x) for x in pml])
        c = None
        if cpml is not None:
            arr = np.asarray(cpml, dtype=np.float64)
            assert arr.size == 6
            c = _dp(arr)
        if self.L.yo_set_boundary(self.h, p, c) != 0:
            raise ValueError("bad pml thickness")

    def set_materials_full(self, eps_r, sigma, mu_r=None):
        e = [np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1)) for a in eps_r]
        s = [np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1)) for a in sigma]
        m = [None] * 3 if mu_r is None else [np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1)) for a in mu_r]
        for a in e + s + [x for x in m if x is not None]:
            assert a.size == self.N
        self.L.yo_set_materials(self.h, *[_dp(a) for a in e], *[_dp(a) for a in s],
                                *[(_dp(a) if a is not None else None) for a in m])

    def set_materials_indexed(self, idx, eps_r, sigma, mu_r=None):
        idx = np.asarray(idx).reshape(-1)
        eps_r = np.asarray(eps_r, dtype=np.float64).reshape(-1, 3)
        sigma = np.asarray(sigma, dtype=np.float64).reshape(-1, 3)
        e = [eps_r[idx, c] for c in range(3)]
        s = [sigma[idx, c] for c in range(3)]
        m = None
        if mu_r is not None:
            mu_r = np.asarray(mu_r, dtype=np.float64).reshape(-1, 3)
            m = [mu_r[idx, c] for c in range(3)]
        self.set_materials_full(e, s, m)

    def add_port(self, port: dict) -> int:
        ints = (C.c_int * 18)(*([int(port.get(k, 0)) for k in _PORT_INT_KEYS] + [0, 0]))
        d = np.array([float(port.get(k, 0.0)) for k in _PORT_DBL_KEYS], dtype=np.float64)
        if port.get("has_source", 0) and "t0" not in port:
            d[1] = 3.0 * d[2]  # t0 = 3 sigma
        r = self.L.yo_add_port(self.h, ints, _dp(d))
        if r < 0:
            raise ValueError("port out of range")
        self.nports = r + 1
        return r

    def set_dft(self, freqs):
        f = np.ascontiguousarray(np.asarray(freqs, dtype=np.float64))
        self.nf = f.size
        self.L.yo_set_dft(self.h, _dp(f), f.size)

    def track_max(self, on=True):
        self.L.yo_set_track_max(self.h, int(on))

    def commit(self):
        self.L.yo_commit(self.h)

    @classmethod
    def from_workload(cls, w: dict, f32=False, track_max=False):
        o = cls(w["nx"], w["ny"], w["nz"], w["dx"], w["dy"], w["dz"], w["dt"], f32=f32,
                periodic_y=bool(w.get("periodic_y", False)))
        o.set_boundary(w["pml"], w.get("cpml"))
        m = w["materials"]
        if m["mode"] == "indexed":
            o.set_materials_indexed(m["idx"], m["eps_r"], m["sigma"], m.get("mu_r"))
        else:
            o.set_materials_full(m["eps_r"], m["sigma"], m.get("mu_r"))
        for p in w.get("ports", []):
            o.add_port(p)
        if len(w.get("freqs", [])):
            o.set_dft(w["freqs"])
        o.track_max(track_max)
        o.commit()
        return o

    # ---- run -----------------------------------------------------------------------------------
    def step(self, n=1):
        r = self.L.yo_step(self.h, int(n))
        if r != 0:
            raise RuntimeError("yo_step before commit")

    @property
    def step_count(self):
        return self.L.yo_step_count(self.h)

    def read_field(self, comp):
        out = np.empty(self.N, dtype=np.float64)
        self.L.yo_read_field(self.h, comp, _dp(out))
        nx, ny, nz = self.shape
        return out.reshape(nz, ny, nx)  # [k, j, i], x fastest

    def write_field(self, comp, arr):
        a = np.ascontiguousarray(np.asarray(arr, dtype=np.float64).reshape(-1))
        assert a.size == self.N
        self.L.yo_write_field(self.h, comp, _dp(a))

    def read_port_dft(self, port):
        V = np.empty(2 * self.nf)
        I = np.empty(2 * self.nf)
        if self.L.yo_read_port_dft(self.h, port, _dp(V), _dp(I)) != 0:
            raise ValueError("bad port")
        return V[0::2] + 1j * V[1::2], I[0::2] + 1j * I[1::2]

    def read_port_last(self, port):
        v = C.c_double()
        i = C.c_double()
        self.L.yo_read_port_last(self.h, port, C.byref(v), C.byref(i))
        return v.value, i.value

    def running_max(self):
        e = C.c_double()
        h = C.c_double()
        self.L.yo_running_max(self.h, C.byref(e), C.byref(h))
        return e.value, h.value

    def cpml_profile(self, axis):
        """R4 coefficient vectors of one axis (0 x, 1 y, 2 z) at every index: dict bE cE ikE (integer positions),
        bH cH ikH (half-integer positions); outside the slabs b = 1, c = 0, 1/kappa = 1."""
        out = {}
        for which, name in enumerate(("bE", "cE", "ikE", "bH", "cH", "ikH")):
            v = np.zeros(self.shape[axis])
            if self.L.yo_cpml_profile(self.h, axis, which, _dp(v)) != 0:
                raise RuntimeError("yo_cpml_profile before commit")
            out[name] = v
        return out

    def psi_norms(self):
        out = np.zeros(12)
        self.L.yo_psi_norms(self.h, _dp(out))
        return out
