"""z-slab decomposition checked on ONE GPU: the slabs of a workload are separate
library handles on the same device, LINKED to each other (fdtd_z_halo / fdtd_z_link): the kernels themselves store the
boundary planes into the neighbour's halo and post / wait on the neighbour's arrival counters, exactly as they do across
GPUs (there the stores travel over NVLink).  The slabs share one stream and advance half step by half step, so every
wait finds its counter already posted by an earlier kernel of the stream: no kernel ever waits for another launch.
Reference: the fp64 oracle on the undivided grid.  fdtd_step(n) of a linked slab (graph replay included) is checked on a
slab linked to ITSELF -- a z-periodic domain -- against the oracle's y-periodic option under the y <-> z mirror map."""
import numpy as np
import pytest

import workloads as W
from oracle.yee import YeeOracle
from paper_2208_04371_b200 import FDTD_F32, FDTD_F64, FDTD_OPT_STEP_IMPL, Solver
from paper_2208_04371_b200.sharded import ShardedSolver

pytestmark = pytest.mark.gpu


def _compare(w, nslabs, steps, tol, dft_tol):
    o = YeeOracle.from_workload(w, track_max=True)
    sh = ShardedSolver(w, ["cuda:0"] * nslabs)
    done = 0
    worst = 0.0
    for cp in (steps // 3, steps):
        o.step(cp - done)
        sh.step(cp - done)
        done = cp
        emax, hmax = o.running_max()
        assert emax > 0 and hmax > 0
        for c in range(6):
            g = sh.read_fields(c).cpu().numpy().astype(np.float64)
            worst = max(worst, np.abs(g - o.read_field(c)).max() / (emax if c < 3 else hmax))
    assert worst <= tol, worst
    vmax = max(np.abs(o.read_port_dft(p)[0]).max() for p in range(len(w["ports"])))
    for p in range(len(w["ports"])):
        Vo, Io = o.read_port_dft(p)
        Vg, Ig = sh.read_port_dft(p)
        assert np.abs(Vo - Vg).max() <= dft_tol * vmax
    return sh


def test_three_slabs_fp32_six_face_cpml():
    """C3's generator at 1/8 scale (192x96x96, CPML on all six faces, ports in the middle slab), three slabs of 32."""
    w = W.throughput_c3(div=8, steps=240, npml=6, nf=16)
    sh = _compare(w, 3, 240, 1e-4, 1e-4)
    # against the undivided GPU run: identical arithmetic except E on the two interface planes (two-pass E kernel there)
    s = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: 2})
    s.step(240)
    for c in range(6):
        a, b = sh.read_fields(c), s.read_fields(c)
        assert float((a - b).abs().max()) <= 2e-5 * float(b.abs().max())
    sh.destroy(); s.destroy()


def test_two_slabs_ground_plane_ports_in_the_lower_slab():
    """C2 at 1/4 scale (128x64x32, z- PEC ground, copper lines, via stub): ports sit on the ground side, slab 0 owns them."""
    w = W.interconnect_c2(run="tot", div=4, steps=600, npml=6, nf=16)
    sh = _compare(w, 2, 600, 1e-4, 1e-4)
    assert all(owner[0] == 0 for owner in sh.owner.values())
    sh.destroy()


def test_two_slabs_fp64_full_coefficients():
    w = W.interconnect_c4(run="tot", div=8, steps=200, npml=5, nf=8)
    assert w["precision"] == FDTD_F64
    sh = _compare(w, 2, 200, 1e-11, 1e-11)
    sh.destroy()


def test_linked_slabs_move_no_plane_from_the_host():
    """The exchange is part of the enqueued kernels: per step a middle slab launches fused + E-on-plane-0 + two waits + two
    posts (+ its port kernels); nothing in ShardedSolver.step copies a plane."""
    import inspect
    from paper_2208_04371_b200 import sharded
    w = W.throughput_c3(div=8, steps=8, npml=6, nf=4)
    sh = ShardedSolver(w, ["cuda:0"] * 3)
    assert not sh.concurrent and len({s.stream.cuda_stream for s in sh.solvers}) == 1
    before = [s.launch_count for s in sh.solvers]
    sh.step(8)
    per_step = [(s.launch_count - b) / 8 for s, b in zip(sh.solvers, before)]
    nport = 1 + sum(1 for p in w["ports"] if p["has_source"])          # k_probe_dft + one k_source per driving port
    assert per_step == [1 + 2, 1 + 1 + 4 + nport, 1 + 1 + 2]           # bottom: no E-plane-0 kernel; the middle slab owns the ports
    assert "copy_" not in inspect.getsource(sharded.ShardedSolver.step)
    sh.destroy()


def _mirror_yz(a):
    """[k, j, i] array of the z-periodic GPU problem -> [j', k', i] array of the y-periodic oracle problem."""
    return np.ascontiguousarray(np.swapaxes(a, 0, 1))


@pytest.mark.parametrize("prec,nsteps", [(FDTD_F64, 19), (FDTD_F32, 26)])
def test_self_linked_slab_steps_with_graphs_like_the_y_periodic_oracle(prec, nsteps):
    """fdtd_step(n) on a linked slab: one handle whose z+ face is linked to its own z- halo and vice versa, i.e. a domain
    periodic in z.  Every wait follows its own post in stream order.  The Yee scheme is invariant under the mirror
    (x, y, z) -> (x, z, y) with E_y <-> E_z, H_x -> -H_x, H_y <-> -H_z, so the oracle's y-periodic option (pinned by the
    parallel-plate tests) on the mirrored inputs is the reference.  Random materials (sigma, mu, anisotropic), CPML on x and
    y, random initial state, no ports."""
    from paper_2208_04371_b200 import FDTD_OPT_GRAPH_UNROLL, binding as B
    wg = W.random_box(41, nx=150, ny=24, nz=20, pml=(4, 3, 3, 4, 0, 0), indexed=False, with_mu=True, steps=nsteps,
                      precision=prec, pec_frac=0.02)
    wg = dict(wg, ports=[], freqs=np.zeros(0))
    m = wg["materials"]
    yz = (0, 2, 1)                                                       # oracle component c holds GPU component yz[c]
    wo = dict(wg, ny=wg["nz"], nz=wg["ny"], dy=wg["dz"], dz=wg["dy"], periodic_y=True,
              pml=[wg["pml"][0], wg["pml"][1], 0, 0, wg["pml"][2], wg["pml"][3]],
              materials={"mode": "full", "eps_r": [_mirror_yz(m["eps_r"][c]) for c in yz],
                         "sigma": [_mirror_yz(m["sigma"][c]) for c in yz], "mu_r": [_mirror_yz(m["mu_r"][c]) for c in yz]})
    r = W.rng_for(4100)
    shape = (wg["nz"], wg["ny"], wg["nx"])
    init = [r.standard_normal(shape) * (1.0 if c < 3 else 2.5e-3) for c in range(6)]
    init[0][:, 0, :] = 0                                                 # walls: j = 0 and i = 0 (z has none here)
    init[1][:, :, 0] = 0
    init[2][:, :, 0] = 0; init[2][:, 0, :] = 0
    o = YeeOracle.from_workload(wo, track_max=True)
    s = Solver.from_workload(wg, precision=prec, options={FDTD_OPT_STEP_IMPL: 2, FDTD_OPT_GRAPH_UNROLL: 4}, z_open=(True, True))
    np_dt = np.float64 if prec == FDTD_F64 else np.float32
    for c in range(3):
        s.write_fields(c, np.ascontiguousarray(init[c], dtype=np_dt))
        s.write_fields(3 + c, np.ascontiguousarray(init[3 + c], dtype=np_dt))
        o.write_field(c, _mirror_yz(init[yz[c]]))
        o.write_field(3 + c, -_mirror_yz(init[3 + yz[c]]))
    # halos of the initial state: plane -1 <- H of the top plane, plane nz <- E of plane 0 (what a previous step would have left)
    import torch
    with torch.cuda.stream(s.stream):
        for comp, src, dst in ((B.FDTD_HX, wg["nz"] - 1, -1), (B.FDTD_HY, wg["nz"] - 1, -1), (B.FDTD_EX, 0, wg["nz"]), (B.FDTD_EY, 0, wg["nz"])):
            s.plane(comp, dst).copy_(s.plane(comp, src))
    for side in (0, 1):                                                  # my z+ pushes into my own z- halo and vice versa
        planes, flag = B.fdtd_z_halo(s.h, 1 - side)
        B.fdtd_z_link(s.h, side, planes, flag)
    o.step(nsteps)
    s.step(nsteps)
    assert s.step_count == nsteps and s.graph_replays == nsteps // 4
    emax, hmax = o.running_max()
    emax = max(emax, max(np.abs(a).max() for a in init[:3]))
    hmax = max(hmax, max(np.abs(a).max() for a in init[3:]))
    worst = 0.0
    for c in range(3):
        ge = s.read_fields(yz[c]).cpu().numpy().astype(np.float64)
        gh = s.read_fields(3 + yz[c]).cpu().numpy().astype(np.float64)
        worst = max(worst, np.abs(_mirror_yz(ge) - o.read_field(c)).max() / emax,
                    np.abs(-_mirror_yz(gh) - o.read_field(3 + c)).max() / hmax)
    assert worst <= (1e-11 if prec == FDTD_F64 else 1e-4), worst
    s.destroy()


def test_a_port_cut_by_an_interface_is_refused():
    w = W.throughput_c3(div=8, steps=10, npml=6, nf=4)          # ports touch planes 45..50; two slabs cut at 48
    with pytest.raises(ValueError, match="cut by a slab interface"):
        ShardedSolver(w, ["cuda:0"] * 2)


def test_slab_handles_refuse_plain_stepping_and_misordered_calls():
    from paper_2208_04371_b200 import FdtdError
    w = W.random_box(5, nx=40, ny=20, nz=24, pml=(3, 3, 3, 3, 0, 0), steps=4, precision=FDTD_F32)
    w = dict(w, ports=[], freqs=np.zeros(0))
    s = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: 2}, z_open=(True, False))
    assert s.impl_name == "fused"
    with pytest.raises(FdtdError):
        s.step(1)                                   # not linked to a neighbour: fdtd_step has no way to fill the halo
    with pytest.raises(FdtdError):
        s.step_end()
    from paper_2208_04371_b200 import binding as B
    with pytest.raises(FdtdError):
        B.fdtd_z_halo(s.h, 1)                       # the z+ face of this slab is a wall, not an interface
    s.step_begin()
    with pytest.raises(FdtdError):
        s.step_begin()
    s.step_end()
    assert s.step_count == 1
    p0, p1 = s.plane(0, -1), s.plane(0, w["nz"])
    assert p0.numel() == p1.numel() > 0
    s.destroy()


def test_linked_slabs_reset_and_run_again_like_a_fresh_run():
    """fdtd_reset of linked slabs (ShardedSolver.reset drains every slab before the first clear and after the last one: a late
    post into a neighbour's counter would satisfy the waits of the next run).  Step, reset, step again: fields and port DFTs
    must be those of a run that never saw the first one, bit for bit."""
    w = W.throughput_c3(div=8, steps=60, npml=6, nf=8)
    sh = ShardedSolver(w, ["cuda:0"] * 3)
    sh.step(37)                                      # an odd count: the ping-pong field sets end up swapped
    sh.reset()
    sh.step(60)
    fresh = ShardedSolver(w, ["cuda:0"] * 3)
    fresh.step(60)
    for c in range(6):
        a, b = sh.read_fields(c), fresh.read_fields(c)
        assert float(b.abs().max()) > 0
        assert bool((a == b).all()), c
    for p in range(len(w["ports"])):
        for x, y in zip(sh.read_port_dft(p), fresh.read_port_dft(p)):
            assert np.array_equal(x, y)
    sh.destroy(); fresh.destroy()


def test_a_wait_that_times_out_is_reported_and_later_waits_return_at_once():
    """A hi-open slab linked to a neighbour that never posts (a scratch buffer stands in for its halo planes and counter), with
    FDTD_OPT_Z_SPIN = 1: the first step's wait is satisfied by the zeroed counter, the second one gives up after one poll and
    sets the slab's time-out flag, every later wait sees the flag and returns without polling; the next synchronising read
    returns FDTD_ECUDA and fdtd_reset clears the condition."""
    import time
    import torch
    from paper_2208_04371_b200 import FdtdError
    from paper_2208_04371_b200 import binding as B
    w = W.random_box(5, nx=40, ny=20, nz=24, pml=(3, 3, 3, 3, 0, 0), steps=4, precision=FDTD_F32)
    w = dict(w, ports=[], freqs=np.zeros(0))
    s = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: 2, B.FDTD_OPT_Z_SPIN: 1}, z_open=(False, True))
    _, nbytes = B.fdtd_plane(s.h, 0, 0)
    dummy = torch.zeros(4 * nbytes + 256, dtype=torch.uint8, device=s.device)    # four planes and a counter nobody posts
    torch.cuda.synchronize()
    base = dummy.data_ptr()
    B.fdtd_z_link(s.h, 1, [base + q * nbytes for q in range(4)], base + 4 * nbytes)
    t0 = time.time()
    s.step(200)
    with pytest.raises(FdtdError) as e:
        s.read_fields(0)
    assert e.value.code == B.FDTD_ECUDA and "timed out" in str(e.value)
    assert time.time() - t0 < 5.0
    s.reset()
    s.step(1)                                        # step 1 waits for "0 steps delivered": satisfied
    s.read_fields(0)
    s.destroy()


@pytest.mark.parametrize("prec", [32, 64])
def test_two_processes_on_one_gpu_exchange_over_cuda_ipc(prec):
    """The cross-process path of f4 on the hardware that exists here: two torch.distributed ranks, both on cuda:0, one z slab
    each, linked through CUDA IPC (DistributedSlab(transport="peer")): the kernels of one process store their boundary planes
    into the other process's halo and post its arrival counter.  Lockstep under host barriers (time-sliced processes); each
    rank checks its slab against the fp64 oracle on the undivided grid, then resets and reruns bit-identically.
    tests/ipc_two_ranks.py is the rank program.  (Two GPUs, concurrent kernels over NVLink: not available on this pool.)"""
    import os
    import socket
    import subprocess
    import sys
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    here = os.path.dirname(os.path.abspath(__file__))
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                        "--master-port", str(port), os.path.join(here, "ipc_two_ranks.py"), str(prec), "60"],
                       capture_output=True, text=True, timeout=600)
    line = [l for l in r.stdout.splitlines() if l.startswith("IPC2 ")]
    print(line[0] if line else r.stdout[-2000:] + r.stderr[-4000:])
    assert r.returncode == 0, r.stderr[-4000:]
    assert line and "rerun_identical=True" in line[0]


def test_slabs_on_two_gpus_match_the_oracle():
    """The path no box of this pool can run (one GPU each): one slab per GPU in one process -- peer access enabled by
    fdtd_z_link, the slabs' kernels running concurrently and waiting on each other's counters over NVLink, fdtd_step(n) with
    graphs on both handles.  Skipped on one GPU; the first box with two runs it."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    w = W.interconnect_c2(run="tot", div=4, steps=600, npml=6, nf=16)
    o = YeeOracle.from_workload(w, track_max=True)
    sh = ShardedSolver(w, ["cuda:0", "cuda:1"])
    assert sh.concurrent
    o.step(600)
    sh.step(600)
    emax, hmax = o.running_max()
    for c in range(6):
        g = sh.read_fields(c).cpu().numpy().astype(np.float64)
        assert np.abs(g - o.read_field(c)).max() <= 1e-4 * (emax if c < 3 else hmax)
    sh.reset()
    sh.step(600)
    again = [sh.read_fields(c) for c in range(6)]
    sh.reset()
    sh.step(600)
    for c in range(6):
        assert bool((sh.read_fields(c) == again[c]).all())
    sh.destroy()
