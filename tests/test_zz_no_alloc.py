"""fdtd_port_probe_noalloc: the port V / I probes (Eq. 4) for callers that cannot allocate device memory.

Who that is: code that wants a probe at a moment when it has no way to get device memory -- a monitor watching a solver that
is busy stepping (an allocation would synchronise the GPU under it), a plug-in in a host program that handed the whole GPU to
its own memory pool at start-up (an allocation fails there), a hook inside a region where allocator calls are forbidden.  The
entry point keeps the hand-over memory of its multi-block reduction in a fixed array inside the library (about 16 KB per GPU,
at most FDTD_NOALLOC_MAX_PORTS = 16 ports per call), so every call on a GPU shares that array and finds the previous call's
contents in it.  What is checked here, through the C ABI:

  * its V and I equal those of the existing path -- the handle's own probe kernel, read with fdtd_read_port_last -- on the same
    fields, within the fp64 parity tolerance of this suite (both reduce in fp64; only the order of the partial sums differs);
  * on TWO calls in a row with different fields in between (the second call starts from the first one's leftovers), and a
    repeat on unchanged fields gives the same bits;
  * a port list longer than the limit is refused with FDTD_ERANGE and a message, before anything is enqueued;
  * the free device memory is the same before and after a call.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide the other tests), and it
builds everything it needs itself, so it passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

import workloads as W
from paper_2208_04371_b200 import FDTD_EZ, FDTD_F32, FDTD_F64, FDTD_HY, FDTD_HZ, FdtdError, Solver
from paper_2208_04371_b200 import binding as B

from .parity_util import TOL


def _workload(precision):
    """C3's generator at 1/8 scale (192 x 96 x 96, CPML on six faces, 4 small ports) plus two wide probe-only ports just
    beside the driven plane: 2800 and 1500 voltage samples, so that the reduction really spans several blocks."""
    w = dict(W.throughput_c3(div=8, steps=64, npml=6, nf=8))
    wide = dict(w["ports"][1], ip=12, vj0=20, vj1=75, vk0=10, vk1=60, lj0=19, lj1=76, lk0=9, lk1=61)
    tall = dict(w["ports"][1], ip=9, vj0=30, vj1=59, vk0=20, vk1=70, lj0=25, lj1=64, lk0=15, lk1=75)
    w["ports"] = list(w["ports"]) + [wide, tall]
    w["precision"] = precision
    return w


@pytest.mark.gpu
@pytest.mark.parametrize("precision", [FDTD_F32, FDTD_F64])
def test_noalloc_probe_matches_the_handle_probe_on_two_calls_in_a_row(precision):
    import torch
    w = _workload(precision)
    nx, ny, nz = w["nx"], w["ny"], w["nz"]
    s = Solver.from_workload(w, device="cuda:0")
    ports = w["ports"]
    VI = torch.full((2 * len(ports),), float("nan"), dtype=torch.float64, device=s.device)
    s.stream.wait_stream(torch.cuda.current_stream(s.device))

    def both(check_memory):
        ref = np.array([s.read_port_last(p) for p in range(len(ports))])        # existing path: [port][V, I]
        f = {c: s.read_fields(c) for c in (FDTD_EZ, FDTD_HY, FDTD_HZ)}          # the fields those were taken from
        s.synchronize()
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info(s.device)[0]
        B.fdtd_port_probe_noalloc(f[FDTD_EZ], f[FDTD_HY], f[FDTD_HZ], precision, nx, ny, nz, w["dy"], w["dz"], ports, VI,
                                  s.stream.cuda_stream)
        s.synchronize()
        if check_memory:
            assert torch.cuda.mem_get_info(s.device)[0] == free0, "the call changed the amount of free device memory"
        got = VI.cpu().numpy().reshape(-1, 2).copy()
        # scale of each sum: the sum of the magnitudes of its terms (what the rounding of a reordered fp64 sum is relative to)
        ez, hy, hz = (f[c].cpu().numpy().astype(np.float64) for c in (FDTD_EZ, FDTD_HY, FDTD_HZ))
        for n, p in enumerate(ports):
            nj = p["vj1"] - p["vj0"] + 1
            vs = w["dz"] / nj * np.abs(ez[p["vk0"]:p["vk1"], p["vj0"]:p["vj1"] + 1, p["ip"]]).sum()
            is_ = w["dz"] * (np.abs(hz[p["lk0"]:p["lk1"] + 1, p["lj1"], p["ip"]]).sum() +
                             np.abs(hz[p["lk0"]:p["lk1"] + 1, p["lj0"] - 1, p["ip"]]).sum()) + \
                w["dy"] * (np.abs(hy[p["lk1"], p["lj0"]:p["lj1"] + 1, p["ip"]]).sum() +
                           np.abs(hy[p["lk0"] - 1, p["lj0"]:p["lj1"] + 1, p["ip"]]).sum())
            assert abs(got[n, 0] - ref[n, 0]) <= TOL[64] * vs, (n, got[n], ref[n])
            assert abs(got[n, 1] - ref[n, 1]) <= TOL[64] * is_, (n, got[n], ref[n])
        return ref, got

    s.step(40)
    ref1, got1 = both(check_memory=False)     # first call on this GPU in this process: includes the one-time address look-up
    assert np.abs(ref1[:, 0]).max() > 0 and np.abs(ref1[:, 1]).max() > 0, "the pulse has not reached the probes: vacuous test"
    s.step(24)
    ref2, got2 = both(check_memory=True)      # second call: starts from the first one's leftovers in the shared array
    assert not np.array_equal(ref1, ref2)
    _, got3 = both(check_memory=True)         # unchanged fields: same bits
    assert np.array_equal(got2, got3)
    s.destroy()


@pytest.mark.gpu
def test_noalloc_probe_refuses_what_its_scratch_cannot_serve():
    import torch
    w = _workload(FDTD_F32)
    nx, ny, nz = w["nx"], w["ny"], w["nz"]
    z = torch.zeros((nz, ny, nx), dtype=torch.float32, device="cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    many = [w["ports"][0]] * (B.FDTD_NOALLOC_MAX_PORTS + 1)
    VI = torch.zeros(2 * len(many), dtype=torch.float64, device="cuda:0")
    VI1 = torch.zeros(2, dtype=torch.float64, device="cuda:0")
    with pytest.raises(FdtdError) as e:
        B.fdtd_port_probe_noalloc(z, z, z, FDTD_F32, nx, ny, nz, w["dy"], w["dz"], many, VI, stream)
    assert e.value.code == B.FDTD_ERANGE and "at most 16" in str(e.value)
    outside = [dict(w["ports"][0], vk1=nz + 1)]
    with pytest.raises(FdtdError) as e:
        B.fdtd_port_probe_noalloc(z, z, z, FDTD_F32, nx, ny, nz, w["dy"], w["dz"], outside, VI1, stream)
    assert e.value.code == B.FDTD_ERANGE
    host = torch.zeros((nz, ny, nx), dtype=torch.float32)          # a host array where device memory is required
    with pytest.raises(FdtdError) as e:
        B.fdtd_port_probe_noalloc(host, z, z, FDTD_F32, nx, ny, nz, w["dy"], w["dz"], many[:1], VI1, stream)
    assert e.value.code == B.FDTD_EINVAL
    # exactly the limit is served
    B.fdtd_port_probe_noalloc(z, z, z, FDTD_F32, nx, ny, nz, w["dy"], w["dz"], many[:-1], VI[:-2], stream)
    torch.cuda.synchronize()
    assert float(VI.abs().max()) == 0.0


def test_noalloc_probe_port_limit_is_checked_on_the_host():
    """No GPU needed: the port count is refused before any pointer is looked at."""
    z = np.zeros((8, 8, 8), dtype=np.float32)
    port = dict(ip=3, vj0=2, vj1=4, vk0=1, vk1=4, lj0=1, lj1=5, lk0=1, lk1=5)
    VI = np.zeros(2 * 17)
    with pytest.raises(FdtdError) as e:
        B.fdtd_port_probe_noalloc(z, z, z, FDTD_F32, 8, 8, 8, 1e-9, 1e-9, [port] * 17, VI, 0)
    assert e.value.code == B.FDTD_ERANGE
