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

NSTEP = 24                 # 12 passes of the two-steps-per-pass kernel
MARGIN = NSTEP + 1
EDGE = 2 * MARGIN + 16     # crop edge: a compared interior of 16 cells where both faces of an axis are artificial


def _crop_workload(w, lo, hi, keep_ports=()):
    """Sub-box [lo, hi) of workload w as a workload of its own; CPML only on crop faces that are real faces.  Ports listed
    in keep_ports must lie inside the box; they are carried over with their coordinates shifted, frequencies kept."""
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
    ports = []
    for n_ in keep_ports:
        q = dict(w["ports"][n_])
        for key, off in (("is", i0), ("ip", i0), ("sj0", j0), ("sj1", j0), ("vj0", j0), ("vj1", j0), ("lj0", j0), ("lj1", j0),
                         ("sk0", k0), ("sk1", k0), ("vk0", k0), ("vk1", k0), ("lk0", k0), ("lk1", k0)):
            q[key] -= off
        ports.append(q)
    return dict(w, nx=i1 - i0, ny=j1 - j0, nz=k1 - k0, pml=pml, materials=mats, ports=ports,
                freqs=w["freqs"] if ports else np.zeros(0))


def _seams(s, w):
    """Per axis (x, y, z): (origin, period) of the tile / chunk seams of the step implementation in use, and the faces of the
    two-step box (None for the other implementations).  Two steps per pass: owned tiles of 120 x 8 cells (fp32: 30 of 32 lanes
    x 4 cells, rows 2..R-2 of R = 11) counted from the box origin, chunks of fdtd_fused_kz() planes from the box's first plane.
    Fused step: tiles of 128 x 14 (tile 1) or 128 x 6 (tile 2) cells and chunks of fdtd_fused_kz() planes, from cell 0.  The
    two-pass kernels have no seams (None)."""
    if s.impl_name == "two_step":
        b = s.two_step_box
        return [(b[0], 120), (b[2], 8), (b[4], s.fused_kz)], b
    if s.impl_name == "fused":
        return [(0, 128), (0, 14 if s.fused_tile == 1 else 6), (0, s.fused_kz)], None
    return [None, None, None], None


def _place(center, n, plo, phi):
    """Start of a crop of EDGE cells around `center` on an axis of n cells.  A crop never cuts a CPML slab: one that would reach
    into a slab is moved flush to that real face instead (it then contains the whole slab and the wall)."""
    lo = center - EDGE // 2
    if lo < plo:
        return 0
    if lo + EDGE > n - phi:
        return n - EDGE
    return int(lo)


def _crops(w, s):
    """Crops whose COMPARED interior (MARGIN cells off every artificial face) holds, for the implementation in use: an x-tile, a
    y-tile and a z-chunk seam at once (two places), each face of the two-step box on each axis (the two corners hold the three
    low / three high faces together with the CPML slabs and walls; three more crops put one high or low face mid-face next to
    seams of the other two axes), the band of one-step cells around a port plane, plus three random interior crops."""
    n = (w["nx"], w["ny"], w["nz"])
    pml = w["pml"]
    seams, box = _seams(s, w)
    r = W.rng_for(990)

    def seam_near(a, frac):
        """a seam of axis a close to frac * n (falls back to that position where the implementation has no seams)"""
        c = int(frac * n[a])
        if seams[a] is None:
            return c
        o, per = seams[a]
        return o + per * max(1, round((c - o) / per))

    def around(cx, cy, cz):
        lo = tuple(_place(c, n[a], pml[2 * a], pml[2 * a + 1]) for a, c in enumerate((cx, cy, cz)))
        return lo, tuple(v + EDGE for v in lo)

    out = [((0, 0, 0), (EDGE,) * 3),                                          # corner: three low CPML slabs + walls (+ box faces)
           (tuple(v - EDGE for v in n), n),                                   # opposite corner: three high slabs
           around(seam_near(0, 0.09), seam_near(1, 0.5), seam_near(2, 0.15)),   # x, y and z seams in one interior (first seams)
           around(seam_near(0, 0.6), seam_near(1, 0.3), seam_near(2, 0.7))]     # ... and deep inside the grid
    seam_checks = [2, 3]
    if box is not None:                                                       # one box face mid-face, seams on the other axes
        out += [around(box[1], seam_near(1, 0.4), seam_near(2, 0.5)),
                around(seam_near(0, 0.4), box[2], seam_near(2, 0.3)),
                around(seam_near(0, 0.7), seam_near(1, 0.6), box[5])]
    else:
        out += [((n[0] - EDGE, 360, 0), (n[0], 360 + EDGE, EDGE))]            # x-high and z-low slabs
    p0 = w["ports"][0]                                                        # the port plane and its band of one-step cells
    out.append(around(p0["ip"], (p0["vj0"] + p0["vj1"]) // 2, (p0["vk0"] + p0["vk1"]) // 2))
    for _ in range(3):                                                        # random interior crops
        o = [int(r.integers(16, m - 16 - EDGE)) for m in n]
        out.append((tuple(o), tuple(v + EDGE for v in o)))
    # the promised seams really lie inside the compared interior
    for q in seam_checks:
        lo, hi = out[q]
        for a in range(3):
            if seams[a] is not None:
                o, per = seams[a]
                inner = range(lo[a] + (MARGIN if lo[a] > 0 else 0) + 1, hi[a] - (MARGIN if hi[a] < n[a] else 0))
                assert any((c - o) % per == 0 for c in inner), (q, a, lo, hi, seams[a])
    return out


@pytest.mark.parametrize("impl,shape", [(0, (1536, 768, 768)), (1, (1536, 768, 768)), (2, (1536, 768, 768)), (4, (1536, 768, 768)),
                                        (0, (2048, 1024, 1024))])
def test_C3_full_size_sampled_subboxes(impl, shape):
    """C3 as benched, and a maximum-size case: 2048x1024x1024 = 2.1 G cells, whose padded arrays (2.19 G elements) pass
    2^31 elements, so every 32-bit offset would show (two field sets + index + psi = 110 GB of the 180 GB)."""
    import torch
    w = W.throughput_c3(steps=NSTEP, shape=shape)
    for q in w["ports"]:
        q["amp"] = 0.0          # the source kernel still runs (bench configuration) but adds nothing: crops carry no ports
    nx, ny, nz = w["nx"], w["ny"], w["nz"]
    s = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: impl})
    # auto picks the fused kernel or two steps per pass at this size, by measurement
    assert s.impl_name in {0: ("fused", "two_step"), 1: ("two_pass",), 2: ("fused",), 4: ("two_step",)}[impl]
    g = torch.Generator(device="cuda").manual_seed(2211)
    init = []
    for c in range(6):
        a = torch.randn((nz, ny, nx), generator=g, device="cuda", dtype=torch.float32) * (1.0 if c < 3 else 2.5e-3)
        if c == 0: a[:, 0, :] = 0; a[0] = 0
        if c == 1: a[:, :, 0] = 0; a[0] = 0
        if c == 2: a[:, :, 0] = 0; a[:, 0, :] = 0
        s.write_fields(c, a)
        init.append(a)
    crops = _crops(w, s)
    init_crops = [[init[c][k0:k1, j0:j1, i0:i1].cpu().numpy().astype(np.float64) for c in range(6)]
                  for (i0, j0, k0), (i1, j1, k1) in crops]
    del init, a
    torch.cuda.empty_cache()
    s.step(NSTEP)
    refs = []
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
        refs.append(([o.read_field(c)[sl] for c in range(6)], sl, emax, hmax))
    worst = 0.0
    for c in range(6):
        full = s.read_fields(c)
        for ((i0, j0, k0), (i1, j1, k1)), (ref, sl, emax, hmax) in zip(crops, refs):
            gpu = full[k0:k1, j0:j1, i0:i1].cpu().numpy().astype(np.float64)
            worst = max(worst, np.abs(gpu[sl] - ref[c]).max() / (emax if c < 3 else hmax))
        del full
    print(f"C3 full size impl={s.impl_name} kz={s.fused_kz} box={s.two_step_box if s.impl_name == 'two_step' else None}: "
          f"{len(crops)} crops of {EDGE}^3, {NSTEP} steps, worst field err {worst:.3e}")
    assert worst <= 1e-4, worst
    s.destroy()


@pytest.mark.parametrize("impl", [0, 2, 4])
def test_C3_full_size_port_probe_and_dft_against_crop_oracle(impl):
    """The probe / DFT path in the configuration the bench runs (1536x768x768, 4 ports, 128 frequencies, the multi-block
    k_probe_dft grid), compared with the oracle at full size: the driven port (source box, V box and I loop) lies inside
    a crop whose artificial faces are further away than the run is long, so the crop oracle's V(t), I(t) and their
    running DFTs equal the full grid's (domain-of-dependence argument above).  Live source plus a random initial
    state, so V and I are O(1) from the first step on.  The run advances two steps per call: with two steps per pass
    (impl 4, or 0 where fdtd_commit selects it) the odd steps' V, I exist only inside the pass -- taken from the band around
    the port plane, with the source the box kernel adds itself -- and are checked through the running DFT."""
    import torch
    nstep = 12
    margin = nstep + 2
    w = W.throughput_c3(steps=nstep)
    nx, ny, nz = w["nx"], w["ny"], w["nz"]
    p0 = w["ports"][0]
    assert p0["has_source"] and len(w["ports"]) == 4 and len(w["freqs"]) == 128
    lo = (16, min(p0["vj0"], p0["lj0"] - 1) - margin, min(p0["vk0"], p0["lk0"] - 1) - margin)
    hi = (p0["ip"] + 1 + margin + 1, max(p0["vj1"], p0["lj1"]) + 1 + margin, max(p0["vk1"], p0["lk1"] + 1) + margin)
    assert p0["ip"] - lo[0] >= margin and p0["is"] - lo[0] >= margin
    s = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: impl})
    assert s.impl_name in {0: ("fused", "two_step"), 2: ("fused",), 4: ("two_step",)}[impl]
    g = torch.Generator(device="cuda").manual_seed(2212)
    (i0, j0, k0), (i1, j1, k1) = lo, hi
    ic = []
    for c in range(6):
        a = torch.randn((nz, ny, nx), generator=g, device="cuda", dtype=torch.float32) * (1.0 if c < 3 else 2.5e-3)
        if c == 0: a[:, 0, :] = 0; a[0] = 0
        if c == 1: a[:, :, 0] = 0; a[0] = 0
        if c == 2: a[:, :, 0] = 0; a[:, 0, :] = 0
        s.write_fields(c, a)
        ic.append(a[k0:k1, j0:j1, i0:i1].cpu().numpy().astype(np.float64))
        del a
    torch.cuda.empty_cache()
    wc = _crop_workload(w, lo, hi, keep_ports=(0,))
    o = YeeOracle.from_workload(wc)
    for c in range(6):
        o.write_field(c, ic[c])
    hist = []
    for _ in range(nstep // 2):
        o.step(2)
        s.step(2)
        hist.append((o.read_port_last(0), s.read_port_last(0)))
    vo, io = np.array([h[0][0] for h in hist]), np.array([h[0][1] for h in hist])
    vg, ig = np.array([h[1][0] for h in hist]), np.array([h[1][1] for h in hist])
    assert np.abs(vo).max() > 0 and np.abs(io).max() > 0
    assert np.abs(vg - vo).max() <= 1e-4 * np.abs(vo).max() and np.abs(ig - io).max() <= 1e-4 * np.abs(io).max()
    Vo, Io = o.read_port_dft(0)
    Vg, Ig = s.read_port_dft(0)
    assert np.abs(Vg - Vo).max() <= 1e-4 * np.abs(Vo).max() and np.abs(Ig - Io).max() <= 1e-4 * np.abs(Io).max()
    # the other three ports run through the same kernel launch; their accumulators must at least be finite and non-zero
    for p in (1, 2, 3):
        v, i = s.read_port_dft(p)
        assert np.isfinite(v).all() and np.isfinite(i).all() and np.abs(v).max() > 0
    s.destroy()
