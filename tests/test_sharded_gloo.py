"""Host-side logic of the z-slab decomposition (paper_2208_04371_b200/sharded.py) without a GPU: the slab plan, the
per-slab workloads and port ownership, and -- with world_size = 2 on the gloo backend -- the two plane exchanges of a
step between neighbouring ranks, driven through DistributedSlab with a stand-in solver that holds CPU planes."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as W
from paper_2208_04371_b200 import sharded as S


def test_plan_covers_the_grid_and_keeps_cpml_in_the_end_slabs():
    for nz, n in ((96, 3), (768, 8), (50, 4), (33, 2)):
        slabs = S.plan_z_slabs(nz, n, 6, 6)
        assert slabs[0][0] == 0 and slabs[-1][1] == nz and all(a[1] == b[0] for a, b in zip(slabs, slabs[1:]))
        assert max(z1 - z0 for z0, z1 in slabs) - min(z1 - z0 for z0, z1 in slabs) <= 1
    with pytest.raises(ValueError):
        S.plan_z_slabs(40, 4, 12, 0)            # the first slab (10 planes) would cut the 12-cell z- layer
    with pytest.raises(ValueError):
        S.plan_z_slabs(10, 4)


def test_shard_workload_slices_materials_moves_ports_and_splits_cpml():
    w = W.throughput_c3(div=8, steps=10, npml=6, nf=4)
    slabs = S.plan_z_slabs(w["nz"], 3, 6, 6)
    seen = []
    for s, (z0, z1) in enumerate(slabs):
        ws, owned = S.shard_workload(w, z0, z1)
        assert ws["nz"] == z1 - z0 and ws["materials"]["idx"].shape[0] == z1 - z0
        assert np.array_equal(ws["materials"]["idx"], w["materials"]["idx"][z0:z1])
        assert ws["pml"][:4] == list(w["pml"][:4])
        assert ws["pml"][4] == (w["pml"][4] if s == 0 else 0) and ws["pml"][5] == (w["pml"][5] if s == 2 else 0)
        for q, n in zip(ws["ports"], owned):
            p = w["ports"][n]
            assert q["vk0"] == p["vk0"] - z0 and q["lk1"] == p["lk1"] - z0 and q["ip"] == p["ip"]
            assert q["lk0"] - 1 >= 0 and q["lk1"] + 1 <= ws["nz"]
        seen += owned
    assert sorted(seen) == list(range(len(w["ports"])))
    assert S.owned_ports(w, 0, 48) == [] and S.owned_ports(w, 48, 96) == []     # two slabs would cut every port


class _FakeSolver:
    """Planes as CPU tensors; begin/end only mark what a real slab would have produced."""
    def __init__(self, ws, rank):
        self.shape = (ws["nz"], ws["ny"], ws["nx"])
        self.device = torch.device("cpu")
        self.rank, self.log = rank, []
        self.planes = {}

    def plane(self, c, k):
        return self.planes.setdefault((c, k), torch.full((64,), float("nan")))

    def step_begin(self):
        self.log.append("begin")
        for c in (S.HX, S.HY):                              # "new H of my top plane"
            self.plane(c, self.shape[0] - 1).fill_(1000.0 * self.rank + 10 * c + len(self.log))

    def step_end(self):
        self.log.append("end")
        for c in (S.EX, S.EY):                              # "new E of my plane 0"
            self.plane(c, 0).fill_(-1000.0 * self.rank - 10 * c - len(self.log))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.interconnect_c2(run="tot", div=4, steps=4, npml=6, nf=4)       # 128x64x32: ports on the ground side
    d = S.DistributedSlab(w, "cpu", make_solver=lambda ws, o, dev, zo: _FakeSolver(ws, rank), transport="nccl")
    d.step(2)
    f = d.solver
    nzl = f.shape[0]
    out[rank] = dict(slab=d.slabs[rank], owner=dict(d.owner), log=list(f.log),
                     halo_lo={c: float(f.plane(c, -1)[0]) for c in (S.HX, S.HY)},
                     halo_hi={c: float(f.plane(c, nzl)[0]) for c in (S.EX, S.EY)})
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_exchange_the_right_planes_in_the_right_order():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        r = dict(out)
    assert r[0]["slab"] == (0, 16) and r[1]["slab"] == (16, 32)
    assert r[0]["owner"] == r[1]["owner"] == {0: (0, 0), 1: (0, 1)}
    assert r[0]["log"] == r[1]["log"] == ["begin", "end", "begin", "end"]
    # rank 1's halo plane -1 holds rank 0's top-plane Hx, Hy as they were after the second begin (log length 3)
    assert r[1]["halo_lo"] == {S.HX: 10.0 * S.HX + 3, S.HY: 10.0 * S.HY + 3}
    # rank 0's halo plane nz holds rank 1's plane-0 Ex, Ey as they were after the second end (log length 4)
    assert r[0]["halo_hi"] == {S.EX: -1000.0 - 10 * S.EX - 4, S.EY: -1000.0 - 10 * S.EY - 4}
    # the outer halos were never written
    assert all(np.isnan(v) for v in r[0]["halo_lo"].values()) and all(np.isnan(v) for v in r[1]["halo_hi"].values())


class _FakeLinkedSolver(_FakeSolver):
    """Stand-in for a slab whose kernels push the planes themselves: export() is what a neighbour needs, link() records
    what this slab was told about a neighbour, step(n) is the only call a linked slab receives."""
    def __init__(self, ws, rank, z_open):
        super().__init__(ws, rank)
        self.z_open, self.links, self.stepped = z_open, {}, []

    def export(self):
        return {"rank": self.rank, "faces": {side: f"halo{side}@{self.rank}" for side, o in enumerate(self.z_open) if o}}

    def link(self, side, nb, exported):
        self.links[side] = (nb, exported["rank"], exported["faces"][1 - side])

    def step(self, n):
        self.stepped.append(n)


def _worker_links(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.throughput_c3(div=8, steps=4, npml=6, nf=4)                     # 192x96x96, ports in the middle slab of three
    d = S.DistributedSlab(w, "cpu", make_solver=lambda ws, o, dev, zo: _FakeLinkedSolver(ws, rank, zo), transport="peer")
    d.step(5)
    out[rank] = dict(links=dict(d.solver.links), stepped=list(d.solver.stepped), log=list(d.solver.log),
                     z_open=d.solver.z_open, owner=dict(d.owner))
    dist.barrier()
    dist.destroy_process_group()


def test_three_ranks_link_to_the_facing_halo_of_each_neighbour_and_step_without_host_exchange():
    world = 3
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker_links, args=(world, _free_port(), out), nprocs=world, join=True)
        r = dict(out)
    assert [r[k]["z_open"] for k in range(3)] == [(False, True), (True, True), (True, False)]
    # side 1 (z+) of rank k is linked to the z- halo (side 0) of rank k+1, side 0 (z-) to the z+ halo (side 1) of rank k-1
    assert r[0]["links"] == {1: (1, 1, "halo0@1")}
    assert r[1]["links"] == {0: (0, 0, "halo1@0"), 1: (2, 2, "halo0@2")}
    assert r[2]["links"] == {0: (1, 1, "halo1@1")}
    # a linked slab is advanced by fdtd_step(n) alone: no begin / end / host-issued exchange
    assert all(r[k]["stepped"] == [5] and r[k]["log"] == [] for k in range(3))
    assert all(r[k]["owner"] == {p: (1, p) for p in range(4)} for k in range(3))


class _FakeResettable(_FakeLinkedSolver):
    """Logs synchronize / reset into a list shared by the ranks; one rank is slow to drain."""
    def __init__(self, ws, rank, z_open, events):
        super().__init__(ws, rank, z_open)
        self.events, self.drains = events, 0

    def synchronize(self):
        import time
        if self.rank == 1 and self.drains == 0:
            time.sleep(0.4)                                   # still finishing its last step while the others are ready to reset
        self.drains += 1
        self.events.append(("sync", self.rank))

    def reset(self):
        self.events.append(("reset", self.rank))


def _worker_reset(rank, world, port, events):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.throughput_c3(div=8, steps=4, npml=6, nf=4)
    d = S.DistributedSlab(w, "cpu", make_solver=lambda ws, o, dev, zo: _FakeResettable(ws, rank, zo, events), transport="peer")
    d.step(3)
    d.reset()
    events.append(("done", rank))
    dist.barrier()
    dist.destroy_process_group()


def test_reset_of_linked_ranks_drains_everybody_before_the_first_clear_and_after_the_last():
    """A neighbour's last kernels store into my halo planes and post my counters: no rank may clear before EVERY rank has
    drained, and no rank may go on (and step) before EVERY rank's clear has landed (include/fdtd.h, fdtd_z_link)."""
    world = 3
    with mp.Manager() as m:
        events = m.list()
        mp.spawn(_worker_reset, args=(world, _free_port(), events), nprocs=world, join=True)
        ev = list(events)
    pos = {kind: [i for i, e in enumerate(ev) if e[0] == kind] for kind in ("sync", "reset", "done")}
    assert len(pos["sync"]) == 2 * world and len(pos["reset"]) == world and len(pos["done"]) == world
    first_syncs = sorted(pos["sync"])[:world]
    assert {ev[i][1] for i in first_syncs} == set(range(world))          # everybody drained ...
    assert max(first_syncs) < min(pos["reset"])                             # ... before the first clear
    assert max(pos["reset"]) < min(pos["done"])                             # and nobody goes on before the last clear
    for r in range(world):                                                  # each rank waits for its own clear to land
        mine = [i for i in pos["sync"] if ev[i][1] == r]
        own_reset = [i for i in pos["reset"] if ev[i][1] == r][0]
        assert mine[0] < own_reset < mine[1]
