"""Parity ladder of the large configs: rungs the oracle can still climb in about a minute.

  C1  full grid, the full 40 000 steps: fp32 fields at the end and S* over the graded 1-500 GHz band (north_star's
      |dS| <= 1e-3); the raw fp32 DFTs are reported against R14's drift, not graded.
  C2  full grid (512x256x128, fp32, indexed), tot run, first 300 steps, in the configuration fdtd_commit selects by itself
      and with the fused kernel forced.
  C4  full grid (1024x512x256, fp64, full anisotropic coefficient arrays, 4 ports, 512 frequencies), first 40 steps:
      fields and raw DFTs to 1e-11.
Rung (ii) of SURVEY 8(d) -- reduced linear scale, FULL step count, S* formed (the method needs 1e5-1e6 steps,
PAPER.md:116; SURVEY G31 flagged S*_11 at 200 k steps in fp32 as the risk):
  C2  1/4 scale (128x64x32), all 200 000 steps, inc + tot (via stub => a real S*_11), fp32 GPU in the configuration commit
      selects and with the fused kernel forced, against the fp64 oracle: fields at 6 checkpoints beside R14's yardstick (the
      oracle's own fp32 instantiation over the same 200 000 steps), S*_11 and S*_21 over the 1-500 GHz band.
  C4  1/8 scale (128x64x32; 1/4 scale = 256x128x64 with FDTD_SLOW=1), all 50 000 steps, inc + tot, fp64 full coefficient
      arrays: fields 1e-11 at 5 checkpoints, raw DFTs 1e-11, S* column formed.
  C3  1/4 scale (384x192x192), all 2000 steps: fields at 5 checkpoints, raw DFTs, S* column.
The oracle is the unmodified fp64 CPU oracle on the same seeded inputs; nothing here comes from the CUDA path.
"""
import os
import numpy as np
import pytest

import workloads as W
from oracle import sparams as osp
from oracle.yee import YeeOracle
from paper_2208_04371_b200 import FDTD_F32, FDTD_F64, FDTD_OPT_STEP_IMPL, Solver, sparams
from tests.parity_util import TOL, assert_fields, run_pair

pytestmark = pytest.mark.gpu
SLOW = os.environ.get("FDTD_SLOW", "0") == "1"


def _sstar(sim, nports, module):
    Vi, Ii = [], []
    for p in range(nports):
        v, i = sim.read_port_dft(p)
        Vi.append(v); Ii.append(i)
    return np.array(module.s_star_column(0, Vi, Ii, Vi))


def test_C1_full_length_sparams():
    w = W.microstrip_c1()          # 192x64x48, 40 000 steps, 128 frequencies 1-500 GHz
    assert w["steps"] == 40000
    o, s, rep = run_pair(w, w["steps"], checkpoints=[2000, 40000])
    assert_fields(rep, FDTD_F32)
    So, Sg = _sstar(o, 2, osp), _sstar(s, 2, sparams)
    dS = np.abs(So - Sg).max()
    print(f"C1 40k steps: field_err={rep['field_err'].max():.3e} dS={dS:.3e} raw dft (V, I) rel err={rep['dft_err']}")
    assert dS <= 1e-3
    assert 0.5 < np.abs(Sg[1]).min() <= np.abs(Sg[1]).max() < 1.5
    # R14: raw fp32 DFTs drift ~1.2e-8 per step against fp64 in the DC-limit band: informational, but it must stay drift-sized
    assert max(rep["dft_err"]) <= 5e-3
    s.destroy()
    # the yardstick of R14 / SURVEY G31: the oracle's own fp32 instantiation (same algorithm, same order) against its fp64
    # run.  The GPU's gap to the fp64 oracle must be of the size of that gap: it is fp32 time stepping, not the kernels.
    from oracle.yee import YeeOracle
    o32 = YeeOracle.from_workload(w, f32=True)
    o32.step(w["steps"])
    vmax = max(np.abs(o.read_port_dft(p)[0]).max() for p in range(2))
    imax = max(np.abs(o.read_port_dft(p)[1]).max() for p in range(2))
    y_v = max(np.abs(o32.read_port_dft(p)[0] - o.read_port_dft(p)[0]).max() for p in range(2)) / vmax
    y_i = max(np.abs(o32.read_port_dft(p)[1] - o.read_port_dft(p)[1]).max() for p in range(2)) / imax
    S32 = _sstar(o32, 2, osp)
    print(f"C1 40k steps, yardstick: fp32 oracle vs fp64 oracle raw dft (V, I) = ({y_v:.3e}, {y_i:.3e}), dS = {np.abs(S32 - So).max():.3e}")
    assert rep["dft_err"][0] <= 2 * y_v + 1e-6 and rep["dft_err"][1] <= 2 * y_i + 1e-6


@pytest.mark.parametrize("impl", [0, 2])
def test_C2_full_grid_first_steps(impl):
    """SURVEY 8(d) rung (i): the full grid, first 500 steps, fields at {100, 250, 500} and the raw port DFTs."""
    w = W.interconnect_c2(run="tot", steps=500)
    assert (w["nx"], w["ny"], w["nz"]) == (512, 256, 128)
    o, s, rep = run_pair(w, 500, options={FDTD_OPT_STEP_IMPL: impl}, checkpoints=[100, 250, 500])
    print(f"C2 full grid 500 steps impl={s.impl_name} kz={s.fused_kz}: field_err={rep['field_err'].max():.3e} dft={rep['dft_err']}")
    assert_fields(rep, FDTD_F32)
    assert max(rep["dft_err"]) <= 1e-4      # 500 steps: far below the drift regime of R14
    s.destroy()


_SLOW = os.environ.get("FDTD_SLOW") == "1"


@pytest.mark.parametrize("impl,steps", [(0, 40), (2, 40)] + ([(0, 500)] if _SLOW else []))
def test_C4_full_grid_first_steps(impl, steps):
    """impl 0: what fdtd_commit selects at this size (the fused step or two steps per pass, by measurement); 2: the fused step.
    40 steps in the default run; rung (i)'s full 500 steps (fields at {100, 250, 500}; about two minutes of fp64 oracle on 134 M
    cells) with FDTD_SLOW=1 -- run once per round through gpurun, its line is kept in profiles/r03_ladder.md."""
    w = W.interconnect_c4(run="tot", steps=steps)
    assert (w["nx"], w["ny"], w["nz"]) == (1024, 512, 256) and w["precision"] == FDTD_F64
    cps = [10, 40] if steps == 40 else [100, 250, 500]
    o, s, rep = run_pair(w, steps, options={FDTD_OPT_STEP_IMPL: impl}, checkpoints=cps)
    print(f"C4 full grid {steps} steps impl={s.impl_name} kz={s.fused_kz}: field_err={rep['field_err'].max():.3e} dft={rep['dft_err']}")
    assert s.impl_name in (("fused", "two_step") if impl == 0 else ("fused",))
    assert_fields(rep, FDTD_F64)
    assert max(rep["dft_err"]) <= 1e-11
    s.destroy()


def test_X3_shaped_full_grid_first_steps():
    """the grid shape and time scale of the paper's CMOS line (200x120x800 cells of (20, 50, 5) nm,
    dt = 0.0145 fs): strongly anisotropic cells, a ragged x tile (200 = 128 + 72), 16 400-sample
    port boxes (multi-block probe reduction), DGAUSS source."""
    w = W.cmos_line_x3(run="tot", steps=150)
    assert (w["nx"], w["ny"], w["nz"]) == (200, 120, 800) and abs(w["dt"] - 0.0145e-15) < 0.00005e-15
    for impl in (0, 2):
        o, s, rep = run_pair(w, 150, options={FDTD_OPT_STEP_IMPL: impl}, checkpoints=[50, 150])
        print(f"X3 full grid impl={s.impl_name} kz={s.fused_kz}: field_err={rep['field_err'].max():.3e} dft={rep['dft_err']}")
        assert_fields(rep, FDTD_F32)
        assert max(rep["dft_err"]) <= 1e-4
        s.destroy()


# ---- rung (ii): reduced scale, full step count, S* ---------------------------------------------------------------------
def _run_to_checkpoints(w, gpu_options, checkpoints, prec):
    """The fp64 oracle and one GPU solver per entry of gpu_options through the same workload; fields compared at every
    checkpoint against the oracle's running maxima (R13).  Returns (oracle, {name: solver}, {name: worst field error})."""
    o = YeeOracle.from_workload(w, track_max=True)
    gpus = {name: Solver.from_workload(w, precision=prec, options=opts) for name, opts in gpu_options.items()}
    worst = {name: 0.0 for name in gpus}
    done = 0
    for cp in checkpoints:
        o.step(cp - done)
        for g in gpus.values():
            g.step(cp - done)
        done = cp
        emax, hmax = o.running_max()
        assert emax > 0 and hmax > 0
        for c in range(6):
            ref = o.read_field(c)
            for name, g in gpus.items():
                d = np.abs(g.read_fields(c).cpu().numpy().astype(np.float64) - ref).max()
                worst[name] = max(worst[name], d / (emax if c < 3 else hmax))
    return o, gpus, worst


def _dfts(sim, nports):
    V, I = zip(*[sim.read_port_dft(p) for p in range(nports)])
    return np.array(V), np.array(I)


def _s_column(inc, tot, nports, module):
    Vi, Ii = _dfts(inc, nports)
    Vt, _ = _dfts(tot, nports)
    return np.array(module.s_star_column(0, list(Vi), list(Ii), list(Vt)))


def _family_errors(sim_fields, o, emax, hmax):
    """max|dE| / running max|E| and max|dH| / running max|H| of a six-component state against the oracle's."""
    e = max(np.abs(sim_fields(c) - o.read_field(c)).max() for c in range(3)) / emax
    h = max(np.abs(sim_fields(c) - o.read_field(c)).max() for c in range(3, 6)) / hmax
    return e, h


def test_C2_quarter_scale_full_200k_steps_sparams():
    """What this rung measures (numbers in profiles/r02_ladder.md): the GAUSS pulse leaves a static charge on the copper
    lines, so E stays at ~0.95 of its running maximum for the rest of the run, and fp32 storage of that static field has
    a frozen rounding pattern whose discrete curl is not zero: H drifts linearly in ANY fp32 time stepping -- the
    oracle's own fp32 instantiation (R14's yardstick, same algorithm and order on the CPU) is 0.4 of max|H| away from
    its fp64 run after 200 000 steps, E 1e-3 of max|E|.  The 1e-4 field bar is therefore asserted while it is reachable
    (the 500-step checkpoint) and, later, the GPU is held to the yardstick: it may not be further from the fp64 oracle
    than a small multiple of what fp32 time stepping itself loses.  S* -- a ratio of DFTs of the same run, Eq. 1 -- is
    graded at the full 200 000 steps against north_star's 1e-3."""
    cps = [500, 2000, 20000, 60000, 120000, 200000]
    opts = {"auto": None}
    if _SLOW:     # the fused step by name as well (the same 200 000 steps again: FDTD_SLOW=1 only; r02_ladder.md has its numbers)
        opts["fused"] = {FDTD_OPT_STEP_IMPL: 2}
    sims = {}
    for run in ("inc", "tot"):
        w = W.interconnect_c2(run=run, div=4)
        assert (w["nx"], w["ny"], w["nz"], w["steps"], len(w["freqs"])) == (128, 64, 32, 200000, 256)
        o = YeeOracle.from_workload(w, track_max=True)
        o32 = YeeOracle.from_workload(w, f32=True)
        gpus = {name: Solver.from_workload(w, options=op) for name, op in opts.items()}
        done = 0
        for cp in cps:
            o.step(cp - done); o32.step(cp - done)
            for g in gpus.values():
                g.step(cp - done)
            done = cp
            emax, hmax = o.running_max()
            ye, yh = _family_errors(o32.read_field, o, emax, hmax)
            line = f"C2/4 {run} step {cp}: fp32-oracle yardstick dE {ye:.2e} dH {yh:.2e};"
            for name, g in gpus.items():
                ge, gh = _family_errors(lambda c: g.read_fields(c).cpu().numpy().astype(np.float64), o, emax, hmax)
                line += f" {name} ({g.impl_name}) dE {ge:.2e} dH {gh:.2e};"
                if cp <= 500:
                    assert max(ge, gh) <= TOL[FDTD_F32], (name, cp, ge, gh)
                assert ge <= 2 * ye + TOL[FDTD_F32] and gh <= 2 * yh + TOL[FDTD_F32], (name, cp, ge, gh, ye, yh)
            print(line)
        sims[run] = (o, gpus, o32)
    So = _s_column(sims["inc"][0], sims["tot"][0], 2, osp)
    # the via stub reflects: S*_11 is a non-zero entry here (about 1.3e-3 in this DC-limit band at 1/4 scale; C1's is identically 0)
    assert np.abs(So[0]).min() > 5e-4, "S*_11 of this test is meant to be non-trivial"
    Vo, Io = _dfts(sims["tot"][0], 2)
    for name in opts:
        Sg = _s_column(sims["inc"][1][name], sims["tot"][1][name], 2, sparams)
        d11, d21 = np.abs(So[0] - Sg[0]).max(), np.abs(So[1] - Sg[1]).max()
        Vg, Ig = _dfts(sims["tot"][1][name], 2)
        raw = (np.abs(Vg - Vo).max() / np.abs(Vo).max(), np.abs(Ig - Io).max() / np.abs(Io).max())
        print(f"C2/4 200k steps {name}: |dS*_11| = {d11:.3e}, |dS*_21| = {d21:.3e} (max|S*_11| = {np.abs(So[0]).max():.3f}, "
              f"max|S*_21| = {np.abs(So[1]).max():.3f}); raw fp32 DFT drift (V, I) = ({raw[0]:.3e}, {raw[1]:.3e}), informational (R14)")
        assert d11 <= 1e-3 and d21 <= 1e-3                      # north_star's bar, absolute
        assert d11 <= 0.05 * np.abs(So[0]).min()                  # and S*_11 itself is resolved, not just below the bar
    S32 = _s_column(sims["inc"][2], sims["tot"][2], 2, osp)
    V32, I32 = _dfts(sims["tot"][2], 2)
    print(f"C2/4 200k steps yardstick (fp32 oracle vs fp64 oracle): |dS*_11| = {np.abs(So[0] - S32[0]).max():.3e}, "
          f"|dS*_21| = {np.abs(So[1] - S32[1]).max():.3e}, raw DFT (V, I) = ({np.abs(V32 - Vo).max() / np.abs(Vo).max():.3e}, "
          f"{np.abs(I32 - Io).max() / np.abs(Io).max():.3e})")
    for _, gpus, _ in sims.values():
        for g in gpus.values():
            g.destroy()


@pytest.mark.parametrize("div", [8] + ([4] if SLOW else []))
def test_C4_reduced_scale_full_50k_steps_fp64(div):
    cps = [500, 5000, 15000, 30000, 50000]
    sims = {}
    for run in ("inc", "tot"):
        w = W.interconnect_c4(run=run, div=div)
        assert (w["steps"], len(w["freqs"]), len(w["ports"]), w["precision"]) == (50000, 512, 4, FDTD_F64)
        o, gpus, worst = _run_to_checkpoints(w, {"auto": None, "fused": {FDTD_OPT_STEP_IMPL: 2}}, cps, FDTD_F64)
        print(f"C4/{div} {run} 50k steps: field_err " + ", ".join(f"{k} ({g.impl_name}) {worst[k]:.3e}" for k, g in gpus.items()))
        assert max(worst.values()) <= TOL[FDTD_F64], worst
        sims[run] = (o, gpus)
    So = _s_column(sims["inc"][0], sims["tot"][0], 4, osp)
    Vo, Io = _dfts(sims["tot"][0], 4)
    for name in ("auto", "fused"):
        Vg, Ig = _dfts(sims["tot"][1][name], 4)
        raw = max(np.abs(Vg - Vo).max() / np.abs(Vo).max(), np.abs(Ig - Io).max() / np.abs(Io).max())
        Sg = _s_column(sims["inc"][1][name], sims["tot"][1][name], 4, sparams)
        dS = np.abs(So - Sg).max()
        print(f"C4/{div} 50k steps {name}: raw DFT {raw:.3e}, |dS*| = {dS:.3e} (max|S*_11| = {np.abs(So[0]).max():.3f})")
        assert raw <= 1e-11 and dS <= 1e-7
    for _, gpus in sims.values():
        for g in gpus.values():
            g.destroy()


def test_C3_quarter_scale_full_2000_steps():
    w = W.throughput_c3(div=4)
    assert (w["nx"], w["ny"], w["nz"], w["steps"], w["pml"]) == (384, 192, 192, 2000, [16] * 6)
    o, gpus, worst = _run_to_checkpoints(w, {"auto": None}, [100, 500, 1000, 1500, 2000], FDTD_F32)
    g = gpus["auto"]
    print(f"C3/4 2000 steps ({g.impl_name}, kz {g.fused_kz}): field_err {worst['auto']:.3e}")
    assert worst["auto"] <= TOL[FDTD_F32]
    So, Sg = _s_column(o, o, 4, osp), _s_column(g, g, 4, sparams)     # one structure: tot == inc
    Vo, Io = _dfts(o, 4)
    Vg, Ig = _dfts(g, 4)
    raw = max(np.abs(Vg - Vo).max() / np.abs(Vo).max(), np.abs(Ig - Io).max() / np.abs(Io).max())
    print(f"C3/4 2000 steps: raw DFT {raw:.3e}, |dS*| = {np.abs(So - Sg).max():.3e}")
    assert raw <= 1e-4 and np.abs(So - Sg).max() <= 1e-3
    g.destroy()
