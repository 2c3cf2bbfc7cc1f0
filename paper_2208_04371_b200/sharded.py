"""Domain decomposition along z: one slab per GPU, two plane exchanges per step (PAPER.md:143, 157:
"decomposing the domain into a number of grids equal to the number of GPUs", guard cells exchanged every step).

The arithmetic is the single-GPU library's, slab by slab (include/fdtd.h "domain decomposition along z"); this module only
does bookkeeping (which planes, which ports, which CPML cells belong to which slab) and moves planes:

    every slab   fdtd_step_begin          fused kernel: H^{n+1/2}, and E^{n+1} except on plane 0 of a lo-open slab
    exchange     Hx, Hy of my top plane   -> halo plane -1 of the slab above          (2 planes up)
    every slab   fdtd_step_end            E^{n+1} on plane 0 of lo-open slabs, source, probes, DFT
    exchange     Ex, Ey of my plane 0     -> halo plane nz of the slab below          (2 planes down)

Planes of slabs with equal nx, ny are contiguous buffers of equal size, so an exchange is one copy per plane: a device
copy when the slabs share a process (`ShardedSolver(devices=[...])`, also how the decomposition is tested on one GPU) or
torch.distributed send/recv over NCCL with one slab per rank (`ShardedSolver.distributed()`; NVLink/NVSwitch peer
transfers, 4 planes of nx*ny words per interface per step: 19 MB for a 1536x768 face against ~50 GB of HBM traffic of
the slab's own step, which is why no overlap machinery is built around it).
"""
from __future__ import annotations

import numpy as np

from . import binding as B
from .solver import Solver

EX, EY, HX, HY = B.FDTD_EX, B.FDTD_EY, B.FDTD_HX, B.FDTD_HY


def plan_z_slabs(nz, nslabs, pml_lo=0, pml_hi=0, min_planes=4):
    """Cut [0, nz) into nslabs contiguous slabs of near-equal thickness; the z- CPML cells must fall into the first slab and
    the z+ cells into the last one.  Returns [(z0, z1), ...]."""
    if nslabs < 1 or nz < nslabs * min_planes:
        raise ValueError(f"cannot cut {nz} planes into {nslabs} slabs of at least {min_planes}")
    cuts = [round(s * nz / nslabs) for s in range(nslabs + 1)]
    if nslabs > 1 and (cuts[1] < pml_lo or cuts[-2] > nz - pml_hi):
        raise ValueError("a z CPML layer would be cut by a slab interface: use fewer slabs")
    return [(cuts[s], cuts[s + 1]) for s in range(nslabs)]


def _port_planes(p):
    """Planes a port touches: (lowest, highest + 1), I loop rows lk0-1 .. lk1 included."""
    lo = min(p["vk0"], p["lk0"] - 1, p["sk0"] if p["has_source"] else p["vk0"])
    hi = max(p["vk1"], p["lk1"] + 1, p["sk1"] if p["has_source"] else p["vk1"])
    return lo, hi


def shard_workload(w, z0, z1):
    """The slab [z0, z1) of workload w as a workload of its own, plus the indices (in w) of the ports it owns.
    A port belongs to the slab that contains all the planes it touches; a port cut by an interface is an error."""
    nz = w["nz"]
    first, last = z0 == 0, z1 == nz
    pml = list(w["pml"])
    pml[4] = pml[4] if first else 0
    pml[5] = pml[5] if last else 0
    m = dict(w["materials"])
    if m["mode"] == "indexed":
        m["idx"] = np.ascontiguousarray(m["idx"][z0:z1])
    else:
        for key in ("eps_r", "sigma", "mu_r"):
            if m.get(key) is not None:
                m[key] = [np.ascontiguousarray(a[z0:z1]) for a in m[key]]
    ports, owned = [], owned_ports(w, z0, z1)
    for n in owned:
        q = dict(w["ports"][n])
        for key in ("vk0", "vk1", "lk0", "lk1", "sk0", "sk1"):
            q[key] -= z0
        ports.append(q)
    return dict(w, nz=z1 - z0, pml=pml, materials=m, ports=ports), owned


def owned_ports(w, z0, z1):
    """Indices of the ports of w that lie inside the slab [z0, z1) with every plane they touch (ports cut by an interface
    belong to no slab; the caller reports them)."""
    return [n for n, p in enumerate(w["ports"]) if _port_planes(p)[0] >= z0 and _port_planes(p)[1] <= z1]


class ShardedSolver:
    """All slabs of a workload.  `devices`: one entry per slab (repeat a device to put several slabs on one GPU)."""

    def __init__(self, w, devices, options=None):
        nsl = len(devices)
        self.w = w
        self.slabs = plan_z_slabs(w["nz"], nsl, w["pml"][4], w["pml"][5])
        self.solvers, self.owner = [], {}
        opts = {B.FDTD_OPT_STEP_IMPL: 2}
        opts.update(options or {})
        for s, ((z0, z1), dev) in enumerate(zip(self.slabs, devices)):
            ws, owned = shard_workload(w, z0, z1)
            for local, n in enumerate(owned):
                self.owner[n] = (s, local)
            z_open = (s > 0, s < nsl - 1)
            self.solvers.append(Solver.from_workload(ws, options=opts, device=dev, z_open=z_open if nsl > 1 else None))
        missing = [n for n in range(len(w["ports"])) if n not in self.owner]
        if missing:
            raise ValueError(f"ports {missing} are cut by a slab interface: choose another number of slabs")

    def _copy(self, src_solver, src, dst_solver, dst):
        """One plane from src_solver's workspace to dst_solver's, ordered after the producer's stream; the producer's next
        kernel waits for the copy (it will overwrite the plane two steps later)."""
        import torch
        done = torch.cuda.Event()
        done.record(src_solver.stream)
        dst_solver.stream.wait_event(done)
        with torch.cuda.device(dst_solver.device), torch.cuda.stream(dst_solver.stream):
            dst.copy_(src, non_blocking=True)
        copied = torch.cuda.Event()
        copied.record(dst_solver.stream)
        src_solver.stream.wait_event(copied)

    def step(self, n=1):
        S = self.solvers
        if len(S) == 1:
            S[0].step(n)
            return
        for _ in range(n):
            for s in S:
                s.step_begin()
            for lo, up in zip(S[:-1], S[1:]):
                top = lo.shape[0] - 1
                for c in (HX, HY):
                    self._copy(lo, lo.plane(c, top), up, up.plane(c, -1))
            for s in S:
                s.step_end()
            for lo, up in zip(S[:-1], S[1:]):
                for c in (EX, EY):
                    self._copy(up, up.plane(c, 0), lo, lo.plane(c, lo.shape[0]))

    def read_fields(self, comp):
        import torch
        return torch.cat([s.read_fields(comp).to(self.solvers[0].device) for s in self.solvers], dim=0)

    def read_port_dft(self, port):
        s, local = self.owner[port]
        return self.solvers[s].read_port_dft(local)

    def synchronize(self):
        for s in self.solvers:
            s.synchronize()

    def destroy(self):
        for s in self.solvers:
            s.destroy()


class DistributedSlab:
    """One slab per torch.distributed rank (backend nccl, one process per GPU).  Same protocol; the copies become
    send/recv pairs between neighbouring ranks.  Port DFTs are read from the owning rank by broadcast."""

    def __init__(self, w, device, options=None, make_solver=None):
        """make_solver(slab_workload, options, device, z_open) -> object with the Solver interface (default: Solver);
        the hook exists so that the exchange protocol can be exercised on CPU tensors under the gloo backend."""
        import torch.distributed as dist
        self.dist, self.rank, self.world = dist, dist.get_rank(), dist.get_world_size()
        self.slabs = plan_z_slabs(w["nz"], self.world, w["pml"][4], w["pml"][5])
        self.owner = {}
        for s, (z0, z1) in enumerate(self.slabs):
            for local, n in enumerate(owned_ports(w, z0, z1)):
                self.owner[n] = (s, local)
        ws, _ = shard_workload(w, *self.slabs[self.rank])
        missing = [n for n in range(len(w["ports"])) if n not in self.owner]
        if missing:
            raise ValueError(f"ports {missing} are cut by a slab interface: choose another number of ranks")
        opts = {B.FDTD_OPT_STEP_IMPL: 2}
        opts.update(options or {})
        z_open = (self.rank > 0, self.rank < self.world - 1)
        make = make_solver or (lambda sw, o, dev, zo: Solver.from_workload(sw, options=o, device=dev, z_open=zo))
        self.solver = make(ws, opts, device, z_open if self.world > 1 else None)
        self.nf = len(w["freqs"])

    def _exchange(self, send_up, comps):
        """send_up: my top plane -> halo plane -1 of rank+1; else my plane 0 -> halo plane nz of rank-1."""
        s, d, ops = self.solver, self.dist, []
        nzl = s.shape[0]
        for c in comps:
            if send_up:
                if self.rank < self.world - 1:
                    ops.append(d.P2POp(d.isend, s.plane(c, nzl - 1), self.rank + 1))
                if self.rank > 0:
                    ops.append(d.P2POp(d.irecv, s.plane(c, -1), self.rank - 1))
            else:
                if self.rank > 0:
                    ops.append(d.P2POp(d.isend, s.plane(c, 0), self.rank - 1))
                if self.rank < self.world - 1:
                    ops.append(d.P2POp(d.irecv, s.plane(c, nzl), self.rank + 1))
        if ops:
            st = getattr(s, "stream", None)          # a CUDA solver runs on its own stream; the collectives on the current one
            if st is not None:
                import torch
                torch.cuda.current_stream(s.device).wait_stream(st)
            for r in d.batch_isend_irecv(ops):
                r.wait()
            if st is not None:
                st.wait_stream(torch.cuda.current_stream(s.device))

    def step(self, n=1):
        if self.world == 1:
            self.solver.step(n)
            return
        for _ in range(n):
            self.solver.step_begin()
            self._exchange(True, (HX, HY))
            self.solver.step_end()
            self._exchange(False, (EX, EY))

    def read_port_dft(self, port):
        import torch
        s, local = self.owner[port]
        buf = torch.zeros(4 * self.nf, dtype=torch.float64, device=self.solver.device)
        if s == self.rank:
            V, I = self.solver.read_port_dft(local)
            buf.copy_(torch.from_numpy(np.concatenate([V.view(np.float64), I.view(np.float64)])))
        self.dist.broadcast(buf, src=s)
        a = buf.cpu().numpy()
        return a[:2 * self.nf].view(np.complex128), a[2 * self.nf:].view(np.complex128)
