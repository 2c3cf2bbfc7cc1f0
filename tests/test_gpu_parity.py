"""Parity of the CUDA path (through the C ABI) with the fp64 CPU oracle, element by element, on seeded inputs.

All tests need a B200: `pytest -m gpu`.  Sizes are chosen so that the oracle finishes in seconds while the grid
still spans several thread blocks / tiles and a ragged tail in every axis.
"""
import math

import numpy as np
import pytest

import workloads as W
from oracle import sparams as osp
from oracle.yee import YeeOracle
from paper_2208_04371_b200 import (FDTD_F32, FDTD_F64, FDTD_OPT_GRAPH_UNROLL, FDTD_OPT_STEP_IMPL, FDTD_OPT_USE_GRAPH,
                                   FdtdError, Solver, sparams)

from .parity_util import IMPLS, TOL, assert_fields, impl_opts, run_pair, solver_or_skip

pytestmark = pytest.mark.gpu

# IMPLS (parity_util): 1 = two-pass kernels, 2 / 26 = fused E+H kernel on its 14-row / 6-row tile, 3 = persistent,
# 4 = two steps per pass on a box + one-step kernels on the shell (skipped where the grid leaves no such box)


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("seed,indexed,with_mu,pml", [
    (1, True, True, (3, 4, 2, 3, 0, 3)),
    (2, False, False, (0, 3, 3, 0, 2, 2)),
    (3, True, False, (2, 2, 2, 2, 2, 2)),
    (4, False, True, (0, 0, 0, 0, 0, 0)),
])
@pytest.mark.parametrize("prec", [FDTD_F64, FDTD_F32])
def test_random_box_every_term(seed, indexed, with_mu, pml, prec, impl):
    """Random eps / sigma / mu blocks, PEC cells, kappa != 1, alpha != 0, mixed CPML faces, driven + passive port."""
    w = W.random_box(seed, indexed=indexed, with_mu=with_mu, pml=pml, steps=60, precision=prec)
    o, s, rep = run_pair(w, 60, precision=prec, options=impl_opts(impl), checkpoints=[1, 2, 17, 60])
    assert_fields(rep, prec)
    dv, di = rep["dft_err"]
    assert max(dv, di) <= (1e-11 if prec == FDTD_F64 else 1e-4)
    for p in range(2):
        vo, io = o.read_port_last(p)
        vg, ig = s.read_port_last(p)
        assert vg == pytest.approx(vo, rel=1e-3 if prec == FDTD_F32 else 1e-9, abs=1e-30 + 1e-5 * abs(vo))
        assert ig == pytest.approx(io, rel=1e-3 if prec == FDTD_F32 else 1e-9, abs=1e-30 + 1e-5 * abs(io))


@pytest.mark.parametrize("impl", IMPLS)
@pytest.mark.parametrize("shape", [(21, 14, 12), (37, 5, 9), (130, 19, 7), (2, 2, 2), (5, 3, 2), (259, 34, 21)])
@pytest.mark.parametrize("prec", [FDTD_F64, FDTD_F32])
def test_ragged_shapes(shape, prec, impl):
    """nx not a multiple of the vector width, tiny grids, several blocks in x with a tail."""
    nx, ny, nz = shape
    pml = tuple(min(3, n // 3) for n in (nx, nx, ny, ny, nz, nz))
    if min(shape) < 6:
        # too small for the generator's port boxes: a bare box with random initial fields instead
        d = (5e-9, 4e-9, 6e-9)
        dt = 0.95 * W.cfl_limit(*d)
        r = W.rng_for(100 + nx)
        one = np.ones((nz, ny, nx))
        w = dict(name="tiny", nx=nx, ny=ny, nz=nz, dx=d[0], dy=d[1], dz=d[2], dt=dt, precision=prec, pml=[0] * 6,
                 cpml=None, materials={"mode": "full", "eps_r": [one * 2.0] * 3, "sigma": [one * 1e3] * 3, "mu_r": None},
                 ports=[], freqs=np.zeros(0), steps=30)
        init = [r.standard_normal((nz, ny, nx)) * (1.0 if c < 3 else 1e-3) for c in range(6)]
        # low-face tangential E is zero by construction (R1)
        init[0][:, 0, :] = 0; init[0][0] = 0
        init[1][:, :, 0] = 0; init[1][0] = 0
        init[2][:, :, 0] = 0; init[2][:, 0, :] = 0
        o, s, rep = run_pair(w, 30, precision=prec, options=impl_opts(impl), init_fields=init)
    else:
        w = W.random_box(7, nx=nx, ny=ny, nz=nz, pml=pml, steps=50, precision=prec)
        o, s, rep = run_pair(w, 50, precision=prec, options=impl_opts(impl), checkpoints=[3, 50])
    assert_fields(rep, prec)


@pytest.mark.parametrize("impl", IMPLS)
def test_P2_exact_discrete_eigenmode_on_gpu(impl):
    """The pin P2 of the oracle, applied to the CUDA path directly (closed form, no oracle in the comparison)."""
    nx, ny, nz = 24, 10, 14
    dx, dy, dz = 5e-9, 4e-9, 6e-9
    dt = 0.9 * W.cfl_limit(dx, dy, dz)
    c0, mu0 = 299792458.0, 4e-7 * math.pi
    m = (1, 2, 1)
    kk = [m[a] * math.pi / (n * d) for a, (n, d) in enumerate([(nx, dx), (ny, dy), (nz, dz)])]
    K = np.array([2 / d * math.sin(k * d / 2) for k, d in zip(kk, (dx, dy, dz))])
    A = np.cross(K, [0.3, -1.0, 0.7])
    k_, j_, i_ = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    kx, ky, kz = kk
    Ex = A[0] * np.cos(kx * (i_ + .5) * dx) * np.sin(ky * j_ * dy) * np.sin(kz * k_ * dz)
    Ey = A[1] * np.sin(kx * i_ * dx) * np.cos(ky * (j_ + .5) * dy) * np.sin(kz * k_ * dz)
    Ez = A[2] * np.sin(kx * i_ * dx) * np.sin(ky * j_ * dy) * np.cos(kz * (k_ + .5) * dz)
    cu = np.cross(K, A)
    Hx = cu[0] * np.sin(kx * i_ * dx) * np.cos(ky * (j_ + .5) * dy) * np.cos(kz * (k_ + .5) * dz)
    Hy = cu[1] * np.cos(kx * (i_ + .5) * dx) * np.sin(ky * j_ * dy) * np.cos(kz * (k_ + .5) * dz)
    Hz = cu[2] * np.cos(kx * (i_ + .5) * dx) * np.cos(ky * (j_ + .5) * dy) * np.sin(kz * k_ * dz)
    f = dt / (2 * mu0)
    s = Solver(nx, ny, nz, dx, dy, dz, dt, FDTD_F64)
    s.set_material_mode(1)
    for opt, val in impl_opts(impl).items():
        s.set_option(opt, val)
    s.commit()
    for c, a in enumerate([Ex, Ey, Ez, f * Hx, f * Hy, f * Hz]):
        s.write_fields(c, np.ascontiguousarray(a))
    wn = 2 / dt * math.asin(c0 * dt / 2 * np.linalg.norm(K))   # Yee dispersion relation
    err = 0.0
    for n in (1, 2, 50, 333):
        s.step(n - s.step_count)
        for c, a in enumerate([Ex, Ey, Ez]):
            err = max(err, np.abs(s.read_fields(c).cpu().numpy() - a * math.cos(wn * n * dt)).max())
    assert err / np.abs(A).max() < 1e-11


@pytest.mark.parametrize("impl", IMPLS)
def test_C0_cavity_full(impl):
    """Config C0 as written: 32^3 fp64 PEC cavity, 2000 steps, fields <= 1e-11 of the running maximum."""
    w = W.cavity_c0()
    o, s, rep = run_pair(w, 2000, options=impl_opts(impl), checkpoints=[100, 500, 1000, 2000])
    assert_fields(rep, FDTD_F64)


def _sstar(sim_inc, sim_tot, nports, module):
    Vi, Ii, Vt = [], [], []
    for p in range(nports):
        v, i = sim_inc.read_port_dft(p)
        Vi.append(v); Ii.append(i)
        Vt.append(sim_tot.read_port_dft(p)[0])
    return np.array(module.s_star_column(0, Vi, Ii, Vt))


@pytest.mark.parametrize("impl", IMPLS)
def test_C1_microstrip_fields_and_sparams(impl):
    """Config C1 geometry at full size, first 1500 steps: fp32 fields, raw DFTs and S* (C1: tot == inc, R22)."""
    w = W.microstrip_c1(steps=1500)
    o, s, rep = run_pair(w, 1500, options=impl_opts(impl), checkpoints=[100, 700, 1500])
    assert_fields(rep, FDTD_F32)
    So = _sstar(o, o, 2, osp)
    Sg = _sstar(s, s, 2, sparams)
    assert np.abs(So - Sg).max() <= 1e-3
    assert np.abs(Sg[0]).max() == 0.0 and 0.5 < np.abs(Sg[1]).min()


@pytest.mark.parametrize("impl", IMPLS)
def test_C2_quarter_scale_inc_tot_sparams(impl):
    """Config C2 at 1/4 linear scale (128x64x32), inc and tot runs, 1200 steps: fields and the S* column."""
    sims = {}
    for run in ("inc", "tot"):
        w = W.interconnect_c2(run=run, div=4, steps=1200, npml=6, nf=32)
        o, s, rep = run_pair(w, 1200, options=impl_opts(impl), checkpoints=[300, 1200])
        assert_fields(rep, FDTD_F32)
        sims[run] = (o, s)
    So = _sstar(sims["inc"][0], sims["tot"][0], 2, osp)
    Sg = _sstar(sims["inc"][1], sims["tot"][1], 2, sparams)
    assert np.abs(So - Sg).max() <= 1e-3


@pytest.mark.parametrize("impl", IMPLS)
def test_C4_eighth_scale_fp64_full_coefficients(impl):
    """Config C4 at 1/8 linear scale (128x64x32), fp64, full anisotropic arrays, 4 ports: 1e-11."""
    w = W.interconnect_c4(run="tot", div=8, steps=400, npml=5, nf=16)
    o, s, rep = run_pair(w, 400, options=impl_opts(impl), checkpoints=[50, 400])
    assert_fields(rep, FDTD_F64)
    assert max(rep["dft_err"]) <= 1e-11


@pytest.mark.parametrize("impl", IMPLS)
def test_C3_small_scale_indexed_six_face_cpml(impl):
    """Config C3's generator at 1/8 linear scale (192x96x96): 64-entry table, six CPML faces, 4 ports, fp32."""
    w = W.throughput_c3(div=8, steps=300, npml=6, nf=16)
    o, s, rep = run_pair(w, 300, options=impl_opts(impl), checkpoints=[20, 300])
    assert_fields(rep, FDTD_F32)
    # the S* column of port 1 over the four ports (one structure: tot == inc, so S*_11 = 0 and the rest are transfer ratios)
    So, Sg = _sstar(o, o, 4, osp), _sstar(s, s, 4, sparams)
    assert np.isfinite(Sg).all() and np.abs(So - Sg).max() <= 1e-3


@pytest.mark.parametrize("impl", IMPLS)
def test_graph_replay_equals_plain_launches(impl):
    """fdtd_step(n) through CUDA-graph replay (unroll 4 + remainder) is bit-identical to one launch per step, and the
    graph really is what ran: Solver owns a real stream, so fdtd_step(27) issues 6 replays of 4 steps + 3 plain steps
    (the persistent kernel, impl 3, has no graph: one cooperative launch covers the whole call)."""
    w = W.random_box(11, nx=40, ny=22, nz=18, steps=27, precision=FDTD_F32)
    out = []
    for graph in (0, 1):
        s = solver_or_skip(w, options=impl_opts(impl, {FDTD_OPT_USE_GRAPH: graph, FDTD_OPT_GRAPH_UNROLL: 4}))
        assert s.stream.cuda_stream != 0
        if graph:
            s.step(27)
        else:
            for _ in range(27):
                s.step(1)
        assert s.step_count == 27
        assert s.graph_replays == (6 if graph and impl != 3 else 0), (impl, graph, s.graph_replays)
        out.append([s.read_fields(c).cpu().numpy() for c in range(6)] + list(s.read_port_dft(0)))
        s.destroy()
    for a, b in zip(*out):
        assert np.array_equal(a, b)


def test_null_stream_runs_plain_launches_with_the_same_result():
    """include/fdtd.h: on the NULL (legacy default) stream no graph can be captured; fdtd_step falls back to plain
    launches there and says so through fdtd_graph_replays."""
    import torch
    w = W.random_box(11, nx=40, ny=22, nz=18, steps=27, precision=FDTD_F32, with_mu=False)
    out = []
    for null in (False, True):
        s = Solver(w["nx"], w["ny"], w["nz"], w["dx"], w["dy"], w["dz"], w["dt"], FDTD_F32)
        s.set_boundary(w["pml"], w["cpml"])
        for p in w["ports"]:
            s.add_port(p)
        s.set_dft(w["freqs"])
        s.set_option(FDTD_OPT_STEP_IMPL, 1)
        s.set_option(FDTD_OPT_GRAPH_UNROLL, 4)
        s.commit("cuda:0", stream=torch.cuda.default_stream() if null else None)
        m = w["materials"]
        s.set_materials_indexed(m["idx"], m["eps_r"], m["sigma"], m.get("mu_r"))
        s.step(27)
        assert (s.stream.cuda_stream == 0) == null and (s.graph_replays == 0) == null
        out.append([s.read_fields(c).cpu().numpy() for c in range(6)])
        s.destroy()
    for a, b in zip(*out):
        assert np.array_equal(a, b)


def test_handle_runs_on_its_own_device_whatever_device_is_current():
    """the library records the device of its workspace at commit and makes it current inside every call.  With
    two GPUs the handle lives on cuda:1 while cuda:0 is current; with one GPU the test checks the recorded ordinal and
    that the caller's current device is left alone."""
    import torch
    from paper_2208_04371_b200 import binding as B
    dev = torch.cuda.device_count() - 1
    w = W.random_box(13, steps=12, precision=FDTD_F32)
    o = YeeOracle.from_workload(w, track_max=True)
    o.step(12)
    torch.cuda.set_device(0)
    s = Solver.from_workload(w, device=f"cuda:{dev}", options={FDTD_OPT_STEP_IMPL: 1})
    assert B.fdtd_device(s.h) == dev and torch.cuda.current_device() == 0
    s.step(12)
    assert torch.cuda.current_device() == 0
    emax, hmax = o.running_max()
    for c in range(6):
        g = s.read_fields(c).cpu().numpy().astype(np.float64)
        assert np.abs(g - o.read_field(c)).max() <= 1e-4 * (emax if c < 3 else hmax)
    s.destroy()


def test_state_errors_of_z_slabs_and_oversized_cpml():
    """profile_step on a z slab and write_fields between step_begin and step_end are refused; the fused step
    asked for by name with more CPML cells than its shared memory holds is an error, not a silent two-pass run."""
    w = W.random_box(14, nx=40, ny=22, nz=18, steps=4, precision=FDTD_F32, pml=(3, 3, 3, 3, 0, 0))
    s = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: 2}, z_open=(False, True))
    with pytest.raises(FdtdError) as e:
        s.profile_step(1)
    assert e.value.code == -3
    s.step_begin()
    with pytest.raises(FdtdError) as e:
        s.write_fields(0, s.read_fields(0))
    assert e.value.code == -3
    s.step_end()
    s.write_fields(0, s.read_fields(0))
    s.destroy()
    big = Solver(200, 16, 16, 1e-9, 1e-9, 1e-9, 1e-18, FDTD_F32)
    big.set_boundary([40, 40, 0, 0, 0, 0])
    big.set_option(FDTD_OPT_STEP_IMPL, 2)
    with pytest.raises(FdtdError) as e:
        big.commit()
    assert e.value.code == -1


def test_reset_and_device_pointers():
    """fdtd_reset zeroes the state; read/write accept device pointers; materials accept a device index array."""
    import torch
    w = W.random_box(12, steps=20, precision=FDTD_F32)
    s = Solver.from_workload(w, materials_on_device=True)
    s.step(20)
    a = [s.read_fields(c).clone() for c in range(6)]
    d0 = s.read_port_dft(0)
    s.reset()
    assert s.step_count == 0
    assert all(float(s.read_fields(c).abs().max()) == 0.0 for c in range(6))
    assert np.abs(s.read_port_dft(0)[0]).max() == 0.0
    s.step(20)
    for c in range(6):
        assert torch.equal(a[c], s.read_fields(c))
    assert np.array_equal(d0[0], s.read_port_dft(0)[0])
    # write from a device tensor, read into a host array
    s.write_fields(2, a[0])
    host = np.empty(a[0].shape, dtype=np.float32)
    s.read_fields(2, out=host)
    assert np.array_equal(host, a[0].cpu().numpy())


def test_error_codes_after_commit():
    s = Solver(8, 8, 8, 1e-9, 1e-9, 1e-9, 1e-18, FDTD_F32)
    s.set_boundary([2] * 6)
    with pytest.raises(FdtdError) as e:
        s.step(1)
    assert e.value.code == -3   # FDTD_ESTATE
    s.commit()
    with pytest.raises(FdtdError) as e:
        s.set_boundary([1] * 6)
    assert e.value.code == -3
    with pytest.raises(FdtdError) as e:
        s.set_materials_full([np.ones(512, np.float32)] * 3, [np.zeros(512, np.float32)] * 3)
    assert e.value.code == -3   # handle is in INDEXED mode
    with pytest.raises(FdtdError) as e:
        s.set_materials_indexed(np.zeros(512, np.uint8), [[1.0, 1.0, -2.0]], [[0.0, 0.0, 0.0]])
    assert e.value.code == -1
    s.step(3)
    # a grid this small is in the two-pass regime; commit keeps whichever of its two drivers it measured faster
    assert s.step_count == 3 and (s.launch_count, s.impl_name) in ((6, "two_pass"), (1, "persistent"))


@pytest.mark.parametrize("prec", [FDTD_F64, FDTD_F32])
@pytest.mark.parametrize("kz", [0, 5, 16])
def test_fused_tiles_chunks_and_odd_step_counts(prec, kz):
    """The fused kernel over several x tiles (nx > 2 tiles of 128 / 64 cells with a ragged tail), several y tiles, z
    chunks that do not divide nz, odd step counts (the state then lives in the second field set) and graph replay."""
    from paper_2208_04371_b200 import FDTD_OPT_FUSED_KZ
    w = W.random_box(21, nx=300, ny=21, nz=23, pml=(5, 6, 4, 3, 2, 5), steps=31, precision=prec)
    o, s, rep = run_pair(w, 31, precision=prec, checkpoints=[1, 2, 3, 13, 31],
                         options={FDTD_OPT_STEP_IMPL: 2, FDTD_OPT_FUSED_KZ: kz, FDTD_OPT_GRAPH_UNROLL: 3})
    assert s.impl_name == "fused"
    assert_fields(rep, prec)
    assert max(rep["dft_err"]) <= (1e-11 if prec == FDTD_F64 else 1e-4)


def test_fused_equals_two_pass_closely():
    """Same arithmetic in the same order: the two step implementations agree to a few ulps of the field maximum."""
    w = W.throughput_c3(div=8, steps=100, npml=6, nf=8)
    out = []
    for impl in (1, 2):
        s = Solver.from_workload(w, options=impl_opts(impl))
        s.step(100)
        out.append([s.read_fields(c).cpu().numpy().astype(np.float64) for c in range(6)])
        s.destroy()
    for c in range(6):
        scale = max(np.abs(out[0][c]).max(), 1e-300)
        assert np.abs(out[0][c] - out[1][c]).max() / scale < 2e-6


def test_fused_result_does_not_depend_on_tile_chunk_or_what_commit_selected():
    """Every cell is advanced by the same operations in the same order whatever tile owns it and whichever block recomputes
    it as halo, so the fused step's result is bit-identical across tile shapes (FDTD_OPT_FUSED_TILE), chunk lengths
    (FDTD_OPT_FUSED_KZ) and the configuration fdtd_commit selects by measurement (which may differ from run to run): the
    auto-selected configuration is reproducible in its RESULT even where its choice is not."""
    from paper_2208_04371_b200 import FDTD_OPT_FUSED_KZ, FDTD_OPT_FUSED_TILE
    w = W.throughput_c3(div=4, steps=40, npml=8, nf=8)
    outs, names = [], []
    for opts in ({FDTD_OPT_FUSED_TILE: 1, FDTD_OPT_FUSED_KZ: 12}, {FDTD_OPT_FUSED_TILE: 2, FDTD_OPT_FUSED_KZ: 7},
                 {FDTD_OPT_FUSED_TILE: 2, FDTD_OPT_FUSED_KZ: 32}, {}, {}):
        s = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: 2, **opts})
        assert s.impl_name == "fused" and s.fused_tile in (1, 2)
        if FDTD_OPT_FUSED_TILE in opts:
            assert (s.fused_tile, s.fused_kz) == (opts[FDTD_OPT_FUSED_TILE], opts[FDTD_OPT_FUSED_KZ])
        names.append((s.fused_tile, s.fused_kz))
        s.step(40)
        outs.append([s.read_fields(c).clone() for c in range(6)] + [torch_dft(s)])
        s.destroy()
    for name, other in zip(names[1:], outs[1:]):
        for a, b in zip(outs[0][:6], other[:6]):
            assert bool((a == b).all()), name
        assert np.array_equal(outs[0][6], other[6]), name


@pytest.mark.parametrize("impl", [2, 26, 3, 4])
def test_repeated_runs_are_bitwise_identical(impl):
    """The fused kernel synchronises its warps with mbarriers only (TMA ring, row-to-row and column hand-over) and the
    persistent kernel with grid barriers: a missing edge in either protocol shows up as run-to-run differences.  Many
    blocks per SM wave, several chunks, CPML on every face; three runs must agree bit for bit (compute-sanitizer is not
    available on this pool)."""
    from paper_2208_04371_b200 import FDTD_OPT_FUSED_KZ
    w = W.throughput_c3(div=4, steps=60, npml=8, nf=8)          # 384x192x192: 3 x 14 x 16 blocks of the fused kernel
    outs = []
    for _ in range(3):
        s = Solver.from_workload(w, options=impl_opts(impl, {FDTD_OPT_FUSED_KZ: 12}))
        s.step(60)
        outs.append([s.read_fields(c).clone() for c in range(6)] + [torch_dft(s)])
        s.destroy()
    for other in outs[1:]:
        for a, b in zip(outs[0][:6], other[:6]):
            assert bool((a == b).all())
        assert np.array_equal(outs[0][6], other[6])


def torch_dft(s):
    v, i = s.read_port_dft(0)
    return np.concatenate([v.view(np.float64), i.view(np.float64)])


@pytest.mark.parametrize("impl", IMPLS)
def test_two_overlapping_sources_and_thick_slabs(impl):
    """Degenerate port set-ups: two driving ports whose source boxes overlap (the sum must not depend on the launch
    order), different waveforms, a port without DFT work next to them; CPML slabs that are thicker than what they leave of
    the grid in y (lo + hi = ny - 2)."""
    w = W.random_box(31, nx=70, ny=18, nz=20, pml=(4, 5, 8, 8, 3, 4), steps=80, precision=FDTD_F32)
    p0 = dict(w["ports"][0])
    extra = dict(p0)
    extra.update({"is": p0["is"], "sj0": p0["sj0"] - 1, "sj1": p0["sj1"], "sk0": p0["sk0"], "sk1": p0["sk1"] + 1,
                  "waveform": 2, "f0": 3.0 / (80 * w["dt"]), "amp": -0.7, "ip": p0["ip"] + 3})
    w = dict(w, ports=[p0, w["ports"][1], extra])
    o, s, rep = run_pair(w, 80, options=impl_opts(impl), checkpoints=[1, 40, 80])
    assert_fields(rep, FDTD_F32)
    assert max(rep["dft_err"]) <= 1e-5
    s.destroy()


# ---- two steps per pass (FDTD_OPT_STEP_IMPL = 4, fdtd_step2.cuh) --------------------------------------------------------
def _random_init(shape, seed):
    r = W.rng_for(seed)
    ini = [r.standard_normal(shape) * (1.0 if c < 3 else 2.5e-3) for c in range(6)]
    ini[0][:, 0, :] = 0; ini[0][0] = 0
    ini[1][:, :, 0] = 0; ini[1][0] = 0
    ini[2][:, :, 0] = 0; ini[2][:, 0, :] = 0
    return ini


@pytest.mark.parametrize("prec", [FDTD_F64, FDTD_F32])
@pytest.mark.parametrize("nsteps", [2, 7, 18])
@pytest.mark.parametrize("mats", ["indexed", "indexed+mu", "full", "full+mu"])
def test_two_step_box_alone_on_a_pec_box(prec, nsteps, mats):
    """No CPML, no ports: the box is the whole grid and k_step2 is the only field kernel (plus the two-pass kernels for the
    odd last step).  Several x tiles (300 = 2 x 120 + 60), y tiles, z chunks that do not divide nz, walls on all six
    faces, random materials and a random initial state: every cell of the grid is compared."""
    from paper_2208_04371_b200 import FDTD_OPT_FUSED_KZ
    w = W.random_box(51, nx=300, ny=40, nz=30, pml=(0,) * 6, indexed=mats.startswith("indexed"), with_mu=mats.endswith("mu"),
                     steps=nsteps, precision=prec)
    w = dict(w, ports=[], freqs=np.zeros(0))
    o, s, rep = run_pair(w, nsteps, precision=prec, options={FDTD_OPT_STEP_IMPL: 4, FDTD_OPT_FUSED_KZ: 7, FDTD_OPT_GRAPH_UNROLL: 4},
                         init_fields=_random_init((30, 40, 300), 77))
    assert s.impl_name == "two_step" and s.graph_replays == nsteps // 4
    assert_fields(rep, prec, tol=(1e-12 if prec == FDTD_F64 else 2e-6))
    s.destroy()


@pytest.mark.parametrize("prec", [FDTD_F64, FDTD_F32])
@pytest.mark.parametrize("shift", [0, 57])
@pytest.mark.parametrize("pml", [(5, 6, 4, 3, 0, 5), (4, 4, 4, 4, 4, 4), (0, 7, 0, 5, 3, 0)])
def test_two_step_box_with_cpml_shell_and_ports(prec, pml, shift):
    """CPML on some or all faces and ports: the box keeps two cells from the layers; the shell (CPML cells and the band
    around them) is advanced by the region launches of the two-pass kernels, whose intermediate values in the band the box
    kernel then overwrites.  shift = 0: the generator's ports next to the x- layer (source plane on the last shell plane or,
    without a layer there, inside the box; probe plane inside the box).  shift = 57: source and probe planes deep inside the
    box (the kernel adds the first step's source itself, the probes of that step read the recomputed band around the port
    plane), a second driving port whose source box overlaps the first one with another waveform, and its probe plane in a
    different vector of the row.  Fields at an even and an odd step count, the probes of BOTH steps of every pair (raw DFTs)."""
    w = W.random_box(54, nx=300, ny=44, nz=40, pml=pml, steps=41, precision=prec)
    if shift:
        ports = [dict(q) for q in w["ports"]]
        ports[0]["is"] += shift
        ports[0]["ip"] += shift + 2
        extra = dict(ports[0])
        extra.update({"sj0": extra["sj0"] - 1, "sk1": extra["sk1"] + 1, "waveform": 2, "f0": 2.0 / (41 * w["dt"]), "amp": -0.6,
                      "ip": extra["ip"] + 3})
        w = dict(w, ports=ports + [extra])
    o, s, rep = run_pair(w, 41, precision=prec, options={FDTD_OPT_STEP_IMPL: 4}, checkpoints=[2, 12, 41])
    assert s.impl_name == "two_step"
    b = s.two_step_box
    V = 4 if prec == FDTD_F32 else 2
    assert b[0] == (-(-(pml[0] + 2) // V) * V if pml[0] else 0)                  # the box is set by the CPML layers alone:
    assert b[2] == (pml[2] + 2 if pml[2] else 0) and b[4] == (pml[4] + 2 if pml[4] else 0)   # ports do not shrink it
    assert_fields(rep, prec, tol=(1e-12 if prec == FDTD_F64 else 1e-5))
    assert max(rep["dft_err"]) <= (1e-11 if prec == FDTD_F64 else 1e-5)
    s.destroy()


def test_two_step_refuses_grids_without_a_box():
    """A grid whose CPML layers leave no 32 x 8 x 8 box is an error for FDTD_OPT_STEP_IMPL = 4, not a silent
    change of implementation; so is a z slab."""
    w = W.random_box(1, steps=4, precision=FDTD_F32)            # 20 x 14 x 12
    with pytest.raises(FdtdError) as e:
        Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: 4})
    assert e.value.code == -1
    w = W.random_box(54, nx=300, ny=44, nz=40, pml=(4, 4, 4, 4, 0, 0), steps=4, precision=FDTD_F32)
    with pytest.raises(FdtdError) as e:
        Solver.from_workload(dict(w, ports=[], freqs=np.zeros(0)), options={FDTD_OPT_STEP_IMPL: 4}, z_open=(False, True))
    assert e.value.code == -1


def test_five_driving_ports_two_step_by_name_is_refused_and_the_automatic_choice_steps_on():
    """The two-step kernel carries at most four driving ports in its parameters.  Asked for by name with five it is an error;
    under the automatic choice (a grid of 8 Mi cells, where two steps per pass is a candidate) the handle simply keeps one of
    the other implementations and matches the oracle."""
    w = W.random_box(61, nx=256, ny=256, nz=128, pml=(4, 4, 4, 4, 4, 4), steps=6, precision=FDTD_F32)
    src = dict(w["ports"][0])
    ports = [dict(src) for _ in range(5)]
    for n, q in enumerate(ports):
        q["is"] = src["is"] + 9 * n
        q["ip"] = src["ip"] + 9 * n
        q["amp"] = 1.0 - 0.1 * n
    w = dict(w, ports=ports)
    with pytest.raises(FdtdError) as e:
        Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: 4})
    assert e.value.code == -1
    o, s, rep = run_pair(w, 6, checkpoints=[2, 6])
    assert s.impl_name in ("fused", "two_pass")
    assert_fields(rep, FDTD_F32)
    assert max(rep["dft_err"]) <= 1e-4
    s.destroy()


@pytest.mark.parametrize("name", ["c2", "c1"])
def test_commit_choice_is_remembered_within_a_process(name):
    """fdtd_commit measures its candidates (step implementation, tile, chunk length); near-equal candidates could come out either
    way and differ in rounding order.  The first verdict for a configuration is kept for the life of the process
    (FDTD_OPT_TUNE_MEMO, default on): every later commit of the same workload runs the same implementation -- and gives the same
    bits -- without measuring again."""
    w = W.interconnect_c2(run="tot", steps=6) if name == "c2" else W.microstrip_c1(steps=6)
    first = Solver.from_workload(w)
    choice, t_first = (first.impl_name, first.fused_kz, first.fused_tile), first.commit_s
    first.step(6)
    ref = [first.read_fields(c).clone() for c in range(6)]
    first.destroy()
    for _ in range(3):
        s = Solver.from_workload(w)
        assert (s.impl_name, s.fused_kz, s.fused_tile) == choice
        t_again = s.commit_s
        s.step(6)
        for c in range(6):
            assert bool((s.read_fields(c) == ref[c]).all())
        s.destroy()
    print(f"{name}: choice {choice}, fdtd_commit {t_first * 1e3:.1f} ms measured, {t_again * 1e3:.1f} ms remembered")
    assert t_again < t_first
