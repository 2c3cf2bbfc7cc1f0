"""`Solver`: a handle plus its torch workspace -- a convenience wrapper over the C-ABI functions of binding.py.

Nothing here computes: setup arguments are marshalled to the library, the workspace is one torch uint8 CUDA tensor and
the solver owns a torch.cuda.Stream of its device (a real stream: fdtd_step replays captured CUDA graphs on it, which the
NULL stream cannot do).  Tensors that cross the boundary are ordered against torch's current stream: device inputs are
waited for before the library reads them, device outputs are handed to the current stream after the library wrote them.
Fields come back as torch CUDA tensors shaped [nz, ny, nx] (x fastest).
"""
from __future__ import annotations

import time

import numpy as np

from . import binding as B


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2208_04371_b200 needs a CUDA device: there is no CPU fallback")
    return torch


class Solver:
    def __init__(self, nx, ny, nz, dx, dy, dz, dt, precision=B.FDTD_F32):
        self.h = B.fdtd_create(nx, ny, nz, dx, dy, dz, dt, precision)
        self.shape = (nz, ny, nx)
        self.precision = precision
        self.nf = 0
        self.nports = 0
        self.workspace = None
        self.z_open = (False, False)

    # ---- setup (before commit) ---------------------------------------------------------------------------------
    def set_boundary(self, pml_cells, cpml=None):
        B.fdtd_set_boundary(self.h, pml_cells, cpml)

    def set_material_mode(self, mode, has_mu=False):
        B.fdtd_set_material_mode(self.h, mode, has_mu)

    def add_port(self, port: dict) -> int:
        pid = B.fdtd_add_port(self.h, port)
        self.nports = pid + 1
        return pid

    def set_dft(self, freqs_hz):
        self.nf = int(np.asarray(freqs_hz).size)
        B.fdtd_set_dft(self.h, freqs_hz)

    def set_option(self, option, value):
        B.fdtd_set_option(self.h, option, value)

    def set_z_interfaces(self, lo_open, hi_open):
        self.z_open = (bool(lo_open), bool(hi_open))
        B.fdtd_set_z_interfaces(self.h, lo_open, hi_open)

    def workspace_bytes(self):
        return B.fdtd_workspace_bytes(self.h)

    def commit(self, device="cuda:0", stream=None):
        """Allocate the workspace on `device` and commit.  `stream`: a torch.cuda.Stream of that device to run on (default:
        a new one owned by this solver)."""
        torch = _torch()
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(self.workspace_bytes(), dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
            self.stream.wait_stream(torch.cuda.current_stream(self.device))   # the allocator may still be clearing the block
            t0 = time.perf_counter()
            B.fdtd_commit(self.h, self.workspace, self.stream.cuda_stream)
            self.commit_s = time.perf_counter() - t0      # wall time of fdtd_commit (tables, clears, commit-time measurements)

    # ---- ordering against torch's current stream for tensors that cross the boundary -------------------------------
    def _before_read_of(self, *tensors):
        """The library is about to read these (device) tensors on its stream: wait for their producers."""
        torch = _torch()
        if any(hasattr(t, "is_cuda") and t.is_cuda for t in tensors):
            self.stream.wait_stream(torch.cuda.current_stream(self.device))

    def _after_write_of(self, *tensors):
        """The library has enqueued writes to these (device) tensors: later work on the current stream waits for them."""
        torch = _torch()
        if any(hasattr(t, "is_cuda") and t.is_cuda for t in tensors):
            torch.cuda.current_stream(self.device).wait_stream(self.stream)

    def _check_field_array(self, a, what):
        nz, ny, nx = self.shape
        B._check_cell_array(a, nx * ny * nz, 8 if self.precision == B.FDTD_F64 else 4, what)

    # ---- after commit ------------------------------------------------------------------------------------------
    def set_materials_indexed(self, idx, eps_r, sigma, mu_r=None):
        nz, ny, nx = self.shape
        n = idx.size if isinstance(idx, np.ndarray) else idx.numel()
        if n != nx * ny * nz:
            raise ValueError(f"material index: {nx * ny * nz} cells expected, got {n}")
        self._before_read_of(idx)
        B.fdtd_set_materials_indexed(self.h, idx, eps_r, sigma, mu_r)

    def set_materials_full(self, eps_r, sigma, mu_r=None):
        nz, ny, nx = self.shape
        self._before_read_of(*eps_r, *sigma, *(mu_r or ()))
        B.fdtd_set_materials_full(self.h, eps_r, sigma, mu_r, n_cells=nx * ny * nz, precision=self.precision)

    def step(self, n=1):
        B.fdtd_step(self.h, n)

    def profile_step(self, n=1):
        return B.fdtd_profile_step(self.h, n)

    @property
    def dtype(self):
        torch = _torch()
        return torch.float64 if self.precision == B.FDTD_F64 else torch.float32

    def read_fields(self, comp, out=None):
        if out is None:
            out = _torch().empty(self.shape, dtype=self.dtype, device=self.device)
        self._check_field_array(out, "read_fields")
        self._before_read_of(out)                   # `out` may still be in use by work queued on the current stream
        B.fdtd_read_fields(self.h, comp, out)
        self._after_write_of(out)
        return out

    def write_fields(self, comp, src):
        self._check_field_array(src, "write_fields")
        self._before_read_of(src)
        B.fdtd_write_fields(self.h, comp, src)

    def read_port_dft(self, port):
        return B.fdtd_read_port_dft(self.h, port, self.nf)

    def read_port_last(self, port):
        return B.fdtd_read_port_last(self.h, port)

    def reset(self):
        B.fdtd_reset(self.h)

    @property
    def step_count(self):
        return B.fdtd_step_count(self.h)

    @property
    def launch_count(self):
        return B.fdtd_launch_count(self.h)

    @property
    def graph_replays(self):
        return B.fdtd_graph_replays(self.h)

    @property
    def impl_name(self):
        return B.fdtd_impl_name(self.h)

    @property
    def fused_kz(self):
        return B.fdtd_fused_kz(self.h)

    @property
    def fused_tile(self):
        return B.fdtd_fused_tile(self.h)

    @property
    def two_step_box(self):
        return B.fdtd_two_step_box(self.h)

    # ---- z-slab stepping (include/fdtd.h "domain decomposition along z") ------------------------------------------
    def step_begin(self):
        B.fdtd_step_begin(self.h)

    def step_end(self):
        B.fdtd_step_end(self.h)

    def plane(self, comp, k):
        """The padded plane k in [-1, nz] of component comp in the current field set, as a uint8 view of the workspace
        (contiguous; equal size and layout on every slab of equal nx, ny)."""
        addr, nbytes = B.fdtd_plane(self.h, comp, k)
        off = addr - self.workspace.data_ptr()
        assert 0 <= off and off + nbytes <= self.workspace.numel()
        return self.workspace[off:off + nbytes]

    def synchronize(self):
        self.stream.synchronize()

    def destroy(self):
        if getattr(self, "h", None):
            B.fdtd_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- a workload dict (workloads/__init__.py) -> a committed solver ------------------------------------------
    @classmethod
    def from_workload(cls, w: dict, precision=None, options=None, device="cuda:0", materials_on_device=False, z_open=None,
                      stream=None):
        prec = precision if precision is not None else w["precision"]
        s = cls(w["nx"], w["ny"], w["nz"], w["dx"], w["dy"], w["dz"], w["dt"], prec)
        if w.get("periodic_y"):
            raise ValueError("periodic-y is an oracle-only option")
        s.set_boundary(w["pml"], w.get("cpml"))
        m = w["materials"]
        has_mu = m.get("mu_r") is not None
        s.set_material_mode(B.FDTD_MAT_INDEXED if m["mode"] == "indexed" else B.FDTD_MAT_FULL, has_mu)
        for p in w.get("ports", []):
            s.add_port(p)
        if len(w.get("freqs", [])):
            s.set_dft(w["freqs"])
        for k, v in (options or {}).items():
            s.set_option(k, v)
        if z_open is not None:
            s.set_z_interfaces(*z_open)
        s.commit(device, stream=stream)
        np_dt = np.float64 if prec == B.FDTD_F64 else np.float32
        if m["mode"] == "indexed":
            idx = np.ascontiguousarray(m["idx"], dtype=np.uint8)
            if materials_on_device:
                idx = _torch().from_numpy(idx).to(s.device)
            s.set_materials_indexed(idx, m["eps_r"], m["sigma"], m.get("mu_r"))
        else:
            conv = lambda xs: None if xs is None else [np.ascontiguousarray(x, dtype=np_dt) for x in xs]
            s.set_materials_full(conv(m["eps_r"]), conv(m["sigma"]), conv(m.get("mu_r")))
        return s
