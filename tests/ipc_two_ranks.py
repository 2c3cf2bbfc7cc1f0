"""Helper of tests/test_gpu_sharded.py::test_two_processes_on_one_gpu_exchange_over_cuda_ipc -- one rank of a 2-rank job whose
ranks both use cuda:0.  Not a test module (pytest does not collect it); launched with torch.distributed.run.

Each rank owns one z slab (DistributedSlab, transport="peer"): the neighbour's halo planes and arrival counter are reached through
a CUDA-IPC mapping of the neighbour's workspace, the fused kernel / the plane-0 E kernel store the boundary planes there and
post the counter (system-scope release), the neighbour's wait kernel acquires it.  The ranks advance in lockstep under host
barriers (DistributedSlab.step_lockstep: processes that share a GPU are time-sliced, a kernel must not wait for a kernel of the
other process).  Every rank runs the fp64 oracle on the UNDIVIDED grid and compares its own slab; rank 0 prints one line.
The process group uses gloo: it carries only the host-side barriers and the exchange of the IPC handles (NCCL refuses two ranks
on one device)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    import torch
    import torch.distributed as dist

    import workloads as W
    from oracle.yee import YeeOracle
    from paper_2208_04371_b200 import FDTD_F64
    from paper_2208_04371_b200.sharded import DistributedSlab

    prec, steps = int(sys.argv[1]), int(sys.argv[2])
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    torch.cuda.set_device(0)
    if prec == 64:
        w = W.interconnect_c4(run="tot", div=8, steps=steps, npml=5, nf=8)
    else:
        w = W.interconnect_c2(run="tot", div=4, steps=steps, npml=6, nf=16)      # ports on the ground side: slab 0 owns them
    sl = DistributedSlab(w, "cuda:0", transport="peer")
    z0, z1 = sl.slabs[rank]
    sl.step_lockstep(steps)
    o = YeeOracle.from_workload(w, track_max=True)
    o.step(steps)
    emax, hmax = o.running_max()
    worst = 0.0
    for c in range(6):
        g = sl.solver.read_fields(c).cpu().numpy().astype(np.float64)
        worst = max(worst, np.abs(g - o.read_field(c)[z0:z1]).max() / (emax if c < 3 else hmax))
    dft = 0.0
    for n, (s, local) in sl.owner.items():
        if s == rank:
            Vo, Io = o.read_port_dft(n)
            Vg, Ig = sl.solver.read_port_dft(local)
            dft = max(dft, np.abs(Vo - Vg).max() / max(np.abs(Vo).max(), 1e-300))
    res = [None] * world
    dist.all_gather_object(res, (rank, worst, dft, sl.solver.launch_count))
    # step, reset (drain - clear - drain across the ranks), step again: the same fields bit for bit
    before = [sl.solver.read_fields(c).clone() for c in range(6)]
    sl.reset()
    sl.step_lockstep(steps)
    same = all(bool((sl.solver.read_fields(c) == before[c]).all()) for c in range(6))
    sames = [None] * world
    dist.all_gather_object(sames, same)
    if rank == 0:
        print("IPC2 " + " ".join(f"rank{r}:field_err={e:.3e},dft_err={d:.3e},launches={l}" for r, e, d, l in res) +
              f" rerun_identical={all(sames)}", flush=True)
    tol = 1e-11 if prec == FDTD_F64 else 1e-4
    ok = all(e <= tol for _, e, _, _ in res) and all(d <= tol for _, _, d, _ in res) and all(sames)
    dist.barrier()
    sl.solver.destroy()
    dist.destroy_process_group()
    sys.exit(0 if ok else 1)


if __name__ == "__main__":
    main()
