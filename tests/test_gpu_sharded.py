"""z-slab decomposition checked on ONE GPU: the slabs of a workload are separate
library handles on the same device that exchange halo planes through the ShardedSolver driver, exactly as they would
across GPUs (there the copy is an NVLink peer copy or an NCCL send/recv).  No kernel waits on another one: the slabs are
stepped one after the other from one process.  Reference: the fp64 oracle on the undivided grid."""
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
        s.step(1)
    with pytest.raises(FdtdError):
        s.step_end()
    s.step_begin()
    with pytest.raises(FdtdError):
        s.step_begin()
    s.step_end()
    assert s.step_count == 1
    p0, p1 = s.plane(0, -1), s.plane(0, w["nz"])
    assert p0.numel() == p1.numel() > 0
    s.destroy()
