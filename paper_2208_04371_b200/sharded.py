"""Domain decomposition along z: one slab per GPU, the halo exchange issued from the kernels (
PAPER.md:143, 157: "decomposing the domain into a number of grids equal to the number of GPUs", guard cells exchanged
every step; Table I: weak scaling at 600^3 cells per GPU).

The arithmetic is the single-GPU library's, slab by slab (include/fdtd.h "domain decomposition along z"); this module only
does bookkeeping (which planes, which ports, which CPML cells belong to which slab) and introduces the slabs to each other:

    link      every slab is given the addresses of its neighbours' halo planes and arrival counters (fdtd_z_halo /
              fdtd_z_link): device pointers within one process, CUDA-IPC mappings of the neighbour's workspace across
              processes (torch's IPC machinery opens them: memory plumbing, not arithmetic).
    step      [wait E from above]  fused kernel: H^{n+1/2} everywhere, E^{n+1} except on plane 0 of a lo-open slab; its
              blocks on the top plane also store Hx, Hy into the upper slab's halo plane -1  [post H up]
              [wait H from below]  E^{n+1} on plane 0, stored also into the lower slab's halo plane nz; source, probes,
              DFT  [post E down]

Four planes of nx*ny words cross an interface per step (19 MB for a 1536x768 face against ~50 GB of HBM traffic of the
slab's own step), as stores of the kernels that compute them: no pack/unpack kernels, no host-issued copies, no collective.
`ShardedSolver` drives all slabs from one process (slabs on one GPU share a stream and advance half step by half step, so
that no wait ever precedes its post in stream order: this is also how the decomposition is tested on one GPU);
`DistributedSlab` is one slab per torch.distributed rank.  With transport="nccl" the planes travel as host-issued
send/recv pairs instead (the fallback when CUDA IPC is not available, and the protocol the gloo CPU test exercises).
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


def link_neighbours(lower, upper):
    """Introduce two adjacent slabs of one process to each other (lower.z+ touches upper.z-)."""
    planes, flag = B.fdtd_z_halo(upper.h, 0)          # where Hx, Hy of lower's top plane must go
    B.fdtd_z_link(lower.h, 1, planes, flag)
    planes, flag = B.fdtd_z_halo(lower.h, 1)          # where Ex, Ey of upper's plane 0 must go
    B.fdtd_z_link(upper.h, 0, planes, flag)


class ShardedSolver:
    """All slabs of a workload in one process.  `devices`: one entry per slab (repeat a device to put several slabs on
    one GPU).  Slabs on the same device share one stream."""

    def __init__(self, w, devices, options=None):
        import torch
        nsl = len(devices)
        self.w = w
        self.slabs = plan_z_slabs(w["nz"], nsl, w["pml"][4], w["pml"][5])
        self.solvers, self.owner = [], {}
        opts = {B.FDTD_OPT_STEP_IMPL: 2}
        opts.update(options or {})
        devs = [torch.device(d) for d in devices]
        self.streams = {}
        for d in devs:
            if d not in self.streams:
                self.streams[d] = torch.cuda.Stream(d)
        # every slab on its own GPU: the slabs run concurrently and fdtd_step(n) may be enqueued slab by slab
        self.concurrent = nsl > 1 and len(self.streams) == nsl
        for s, ((z0, z1), dev) in enumerate(zip(self.slabs, devs)):
            ws, owned = shard_workload(w, z0, z1)
            for local, n in enumerate(owned):
                self.owner[n] = (s, local)
            z_open = (s > 0, s < nsl - 1)
            self.solvers.append(Solver.from_workload(ws, options=opts, device=dev, z_open=z_open if nsl > 1 else None,
                                                     stream=self.streams[dev]))
        missing = [n for n in range(len(w["ports"])) if n not in self.owner]
        if missing:
            raise ValueError(f"ports {missing} are cut by a slab interface: choose another number of slabs")
        for lo, up in zip(self.solvers[:-1], self.solvers[1:]):
            link_neighbours(lo, up)

    def step(self, n=1, chunk=8):
        S = self.solvers
        if len(S) == 1:
            S[0].step(n)
        elif self.concurrent:
            # one GPU per slab: enqueue a few steps per slab in turn (a stream that waits for a neighbour must not fill the
            # launch queue before that neighbour's work has been enqueued)
            while n > 0:
                m = min(n, chunk)
                for s in S:
                    s.step(m)
                n -= m
        else:
            # slabs that share a stream: all first halves, then all second halves, in ascending order -- every wait
            # kernel then finds its counter already posted by an earlier kernel of the same stream
            for _ in range(n):
                for s in S:
                    s.step_begin()
                for s in S:
                    s.step_end()

    def read_fields(self, comp):
        import torch
        return torch.cat([s.read_fields(comp).to(self.solvers[0].device) for s in self.solvers], dim=0)

    def upload_materials(self, pinned=False):
        """(Re)send every slab's slice of the indexed material map from host memory; returns the bytes sent."""
        import torch
        m, sent = self.w["materials"], 0
        for s, (z0, z1) in zip(self.solvers, self.slabs):
            idx = torch.from_numpy(np.ascontiguousarray(m["idx"][z0:z1], dtype=np.uint8))
            s.set_materials_indexed(idx.pin_memory() if pinned else idx, m["eps_r"], m["sigma"], m.get("mu_r"))
            sent += idx.numel()
        return sent

    def reset(self):
        """Zero every slab.  Linked slabs write into each other (halo planes, arrival counters), and one slab may be a step
        ahead of its neighbour: all of them must have drained before the first one clears its counters, and all clears must
        have landed before anyone steps again (include/fdtd.h, fdtd_z_link)."""
        self.synchronize()
        for s in self.solvers:
            s.reset()
        self.synchronize()

    @property
    def launch_count(self):
        return sum(s.launch_count for s in self.solvers)

    def read_port_dft(self, port):
        s, local = self.owner[port]
        return self.solvers[s].read_port_dft(local)

    def synchronize(self):
        for s in self.solvers:
            s.synchronize()

    def destroy(self):
        for s in self.solvers:
            s.destroy()


def _ipc_export(solver):
    """What a neighbouring rank needs to write into this slab: a picklable handle of the workspace (CUDA IPC through torch's
    tensor-sharing machinery) and the byte offsets of the halo planes and arrival counters inside it."""
    from torch.multiprocessing.reductions import reduce_tensor
    base = solver.workspace.data_ptr()
    faces = {}
    for side, is_open in enumerate(solver.z_open):
        if is_open:
            planes, flag = B.fdtd_z_halo(solver.h, side)
            faces[side] = ([p - base for p in planes], flag - base)
    return reduce_tensor(solver.workspace), faces


def _ipc_link(solver, side, exported, keep):
    """Map the neighbour's workspace into this process and link `side` of this slab to the neighbour's facing halo."""
    (rebuild, args), faces = exported
    ws = rebuild(*args)
    keep.append(ws)                                   # the mapping must outlive the handle
    planes, flag = faces[1 - side]                    # my z+ touches the neighbour's z-, and the other way round
    B.fdtd_z_link(solver.h, side, [ws.data_ptr() + o for o in planes], ws.data_ptr() + flag)


class DistributedSlab:
    """One slab per torch.distributed rank (one process per GPU).  transport="peer": the slabs are linked through CUDA IPC
    and the kernels push the planes themselves (fdtd_step(n) per rank, no per-step host work); transport="nccl": send/recv
    pairs between neighbouring ranks around fdtd_step_begin / fdtd_step_end.  Port DFTs are read from the owning rank by
    broadcast."""

    def __init__(self, w, device, options=None, make_solver=None, transport="peer"):
        """make_solver(slab_workload, options, device, z_open) -> object with the Solver interface (default: Solver);
        the hook exists so that the exchange protocol can be exercised on CPU tensors under the gloo backend."""
        import torch.distributed as dist
        self.dist, self.rank, self.world = dist, dist.get_rank(), dist.get_world_size()
        self.transport = transport
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
        self._mapped = []
        if transport == "peer" and self.world > 1:
            self._link_over_ipc(make_solver is None)

    def _link_over_ipc(self, real):
        """Every rank publishes its export, then links to rank-1 and rank+1.  `real` is False under the CPU test hook, whose
        solver object supplies export() / link(side, exported) itself."""
        export = _ipc_export(self.solver) if real else self.solver.export()
        everyone = [None] * self.world
        self.dist.all_gather_object(everyone, export)
        for side, nb in ((0, self.rank - 1), (1, self.rank + 1)):
            if 0 <= nb < self.world:
                if real:
                    _ipc_link(self.solver, side, everyone[nb], self._mapped)
                else:
                    self.solver.link(side, nb, everyone[nb])
        self.dist.barrier()                          # nobody steps before everybody is linked

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
        if self.world == 1 or self.transport == "peer":
            self.solver.step(n)                      # linked slabs: the hand-over is inside the enqueued kernels
            return
        for _ in range(n):
            self.solver.step_begin()
            self._exchange(True, (HX, HY))
            self.solver.step_end()
            self._exchange(False, (EX, EY))

    def step_lockstep(self, n=1):
        """n steps with a host barrier after every half step -- for ranks that SHARE one GPU (time-sliced processes: a kernel
        of one process must never spin on a counter that only a kernel of another process can post, the GPU may not be running
        that process).  The hand-over itself is unchanged: the kernels store the planes into the neighbour's halo (CUDA-IPC
        mapped memory) and post its counter; the barriers only make sure every wait finds its counter already posted."""
        for _ in range(n):
            self.solver.step_begin()
            self.solver.synchronize()
            self.dist.barrier()
            self.solver.step_end()
            self.solver.synchronize()
            self.dist.barrier()

    def upload_materials(self, w, pinned=False):
        import torch
        m = w["materials"]
        z0, z1 = self.slabs[self.rank]
        idx = torch.from_numpy(np.ascontiguousarray(m["idx"][z0:z1], dtype=np.uint8))
        self.solver.set_materials_indexed(idx.pin_memory() if pinned else idx, m["eps_r"], m["sigma"], m.get("mu_r"))
        return idx.numel()

    def reset(self):
        """Quiesce, clear, quiesce: a neighbour's last kernels store into my halo planes and post my counters, so every rank
        drains its stream before anyone clears, and every clear has landed on the device before anyone steps again."""
        sync = getattr(self.solver, "synchronize", None)   # the CPU test hook's solver has no stream
        if sync:
            sync()
        self.dist.barrier()                          # everybody's kernels (and their stores into my halo) are done
        self.solver.reset()
        if sync:
            sync()
        self.dist.barrier()                          # nobody posts into a neighbour that has not yet zeroed its counters

    @property
    def launch_count(self):
        return self.solver.launch_count

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
