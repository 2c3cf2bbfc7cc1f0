"""Parity at BASELINE.json's full C3 size (1536x768x768, fp32, uint8 index, six-face CPML), in the launch configuration
bench.py times, on sampled sub-boxes the oracle can compute.

The explicit scheme has a finite numerical domain of dependence: the state of a cell after n steps depends only on the
initial state, the materials and the sources within n cells of it (R5: every half step reaches one neighbour).  So the
oracle, run on a CROP of the full problem (same materials, same initial fields, PEC on the artificial crop faces), equals
the full-grid result on every cell further than n cells from an artificial face.  Crops that touch a real face keep that
face's CPML; crops never cut through a CPML slab.  The initial state is seeded random noise (torch generator on the
device; wall rows zeroed as R1 requires), so every term of the update is exercised at every sampled cell.
"""
import numpy as np
import pytest

import workloads as W
from oracle.yee import YeeOracle
from paper_2208_04371_b200 import FDTD_OPT_STEP_IMPL, Solver

pytestmark = pytest.mark.gpu

NSTEP = 6
MARGIN = NSTEP + 1


def _crop_workload(w, lo, hi):
    """Sub-box [lo, hi) of workload w as a workload of its own; CPML only on crop faces that are real faces."""
    (i0, j0, k0), (i1, j1, k1) = lo, hi
    n = (w["nx"], w["ny"], w["nz"])
    pml = []
    for a, (l, h) in enumerate(zip(lo, hi)):
        pml += [w["pml"][2 * a] if l == 0 else 0, w["pml"][2 * a + 1] if h == n[a] else 0]
        # a crop must not cut through a slab
        assert l == 0 or l >= w["pml"][2 * a], "crop cuts the low slab"
        assert h == n[a] or h <= n[a] - w["pml"][2 * a + 1], "crop cuts the high slab"
    m = w["materials"]
    mats = dict(m)
    mats["idx"] = np.ascontiguousarray(m["idx"][k0:k1, j0:j1, i0:i1])
    return dict(w, nx=i1 - i0, ny=j1 - j0, nz=k1 - k0, pml=pml, materials=mats, ports=[], freqs=np.zeros(0))


def _crops(w):
    nx, ny, nz = w["nx"], w["ny"], w["nz"]
    e = 40  # crop edge; compared interior = e - 2*MARGIN where both faces are artificial
    r = W.rng_for(990)
    out = [((0, 0, 0), (e, e, e)),                                     # corner: three low CPML slabs + walls
           ((nx - e, ny - e, nz - e), (nx, ny, nz)),                   # opposite corner: three high slabs
           ((108, 0, 300), (148, e, 340)),                             # x-tile boundary at i = 128, y-low slab
           ((nx - e, 360, 0), (nx, 400, e)),                           # x-high and z-low slabs, y-tile boundaries
           ((620, 376, 108), (660, 416, 148))]                         # interior: z-chunk boundary at k = 128
    for _ in range(3):                                                 # random interior crops
        o = [int(r.integers(16, n - 16 - e)) for n in (nx, ny, nz)]
        out.append((tuple(o), tuple(v + e for v in o)))
    return out


@pytest.mark.parametrize("impl,shape", [(0, (1536, 768, 768)), (1, (1536, 768, 768)), (0, (2048, 1024, 1024))])
def test_C3_full_size_sampled_subboxes(impl, shape):
    """C3 as benched, and a maximum-size case: 2048x1024x1024 = 2.1 G cells, whose padded arrays (2.19 G elements) pass
    2^31 elements, so every 32-bit offset would show (two field sets + index + psi = 110 GB of the 180 GB)."""
    import torch
    w = W.throughput_c3(steps=NSTEP, shape=shape)
    for q in w["ports"]:
        q["amp"] = 0.0          # the source kernel still runs (bench configuration) but adds nothing: crops carry no ports
    nx, ny, nz = w["nx"], w["ny"], w["nz"]
    s = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: impl})
    assert s.impl_name == ("fused" if impl == 0 else "two_pass")      # auto picks the fused kernel at this size
    g = torch.Generator(device="cuda").manual_seed(2211)
    init = []
    for c in range(6):
        a = torch.randn((nz, ny, nx), generator=g, device="cuda", dtype=torch.float32) * (1.0 if c < 3 else 2.5e-3)
        if c == 0: a[:, 0, :] = 0; a[0] = 0
        if c == 1: a[:, :, 0] = 0; a[0] = 0
        if c == 2: a[:, :, 0] = 0; a[:, 0, :] = 0
        s.write_fields(c, a)
        init.append(a)
    crops = _crops(w)
    init_crops = [[init[c][k0:k1, j0:j1, i0:i1].cpu().numpy().astype(np.float64) for c in range(6)]
                  for (i0, j0, k0), (i1, j1, k1) in crops]
    del init, a
    torch.cuda.empty_cache()
    s.step(NSTEP)
    worst = 0.0
    for (lo, hi), ic in zip(crops, init_crops):
        wc = _crop_workload(w, lo, hi)
        o = YeeOracle.from_workload(wc, track_max=True)
        for c in range(6):
            o.write_field(c, ic[c])
        o.step(NSTEP)
        emax, hmax = o.running_max()
        emax = max(emax, max(np.abs(a).max() for a in ic[:3]))
        hmax = max(hmax, max(np.abs(a).max() for a in ic[3:]))
        (i0, j0, k0), (i1, j1, k1) = lo, hi
        # interior of the crop: MARGIN cells away from every artificial face
        sl = tuple(slice(MARGIN if l > 0 else 0, (h - l) - (MARGIN if h < n else 0))
                   for l, h, n in ((k0, k1, nz), (j0, j1, ny), (i0, i1, nx)))
        for c in range(6):
            gpu = s.read_fields(c)[k0:k1, j0:j1, i0:i1].cpu().numpy().astype(np.float64)
            d = np.abs(gpu[sl] - o.read_field(c)[sl]).max() / (emax if c < 3 else hmax)
            worst = max(worst, d)
    assert worst <= 1e-4, worst
    s.destroy()
