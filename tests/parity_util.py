"""Shared helper of the GPU parity tests: run one workload through the oracle and through the C ABI, compare.

Tolerances (BASELINE.json north_star):
  fields   max|dE|, max|dH| <= 1e-4 of the running field maximum (fp32 GPU), <= 1e-11 (fp64 GPU)          (R13)
  port DFT raw V^, I^ relative to max|.| over the band: 1e-11 (fp64); fp32 is informational (R14) except where stated
"""
import numpy as np

import pytest

from oracle.yee import YeeOracle
from paper_2208_04371_b200 import FDTD_F64, FDTD_OPT_FUSED_TILE, FDTD_OPT_STEP_IMPL, FdtdError, Solver

TOL = {32: 1e-4, 64: 1e-11}

# Step implementations the parity tests run through: FDTD_OPT_STEP_IMPL 1 = two-pass kernels, 2 = fused E+H kernel (TMA-staged,
# ping-pong field sets) on its 14-row tile, 3 = persistent, 4 = two steps per pass on a box + one-step kernels on the shell
# (skipped where the grid leaves no such box); 26 = the fused kernel on its 6-row tile (FDTD_OPT_FUSED_TILE = 2: two blocks
# per SM, the mid-size-grid build).
IMPLS = [1, 2, 3, 4, 26]


def impl_opts(impl, more=None):
    """fdtd_set_option dictionary of a test's step implementation id (IMPLS) plus further options."""
    o = {FDTD_OPT_STEP_IMPL: 2, FDTD_OPT_FUSED_TILE: 2} if impl == 26 else \
        {FDTD_OPT_STEP_IMPL: 2, FDTD_OPT_FUSED_TILE: 1} if impl == 2 else {FDTD_OPT_STEP_IMPL: impl}
    o.update(more or {})
    return o


def solver_or_skip(w, precision=None, options=None, **kw):
    """Solver.from_workload; the two-steps-per-pass implementation (FDTD_OPT_STEP_IMPL = 4) refuses grids that leave no box
    two cells away from the CPML layers and the port planes (FDTD_EINVAL): such a case is skipped, not failed."""
    try:
        return Solver.from_workload(w, precision=precision, options=options, **kw)
    except FdtdError as e:
        if (options or {}).get(FDTD_OPT_STEP_IMPL) == 4 and e.code == -1:
            pytest.skip(f"no two-step box on this grid: {e}")
        raise


def run_pair(w, steps, precision=None, options=None, checkpoints=None, init_fields=None):
    """Returns (oracle, solver, report) after `steps` steps; report['field_err'][c] is the worst relative error over
    the checkpoints (relative to the oracle's running maximum of |E| resp. |H| at that checkpoint)."""
    prec = precision or w["precision"]
    s = solver_or_skip(w, precision=prec, options=options)
    o = YeeOracle.from_workload(w, track_max=True)
    if init_fields is not None:
        for c, a in enumerate(init_fields):
            o.write_field(c, a)
            s.write_fields(c, np.ascontiguousarray(a, dtype=np.float64 if prec == FDTD_F64 else np.float32))
    cps = sorted(set(checkpoints or [steps]))
    assert cps[-1] == steps
    err = np.zeros(6)
    done = 0
    for cp in cps:
        o.step(cp - done)
        s.step(cp - done)
        done = cp
        emax, hmax = o.running_max()
        if init_fields is not None:
            emax = max(emax, max(np.abs(a).max() for a in init_fields[:3]))
            hmax = max(hmax, max(np.abs(a).max() for a in init_fields[3:]))
        for c in range(6):
            scale = emax if c < 3 else hmax
            g = s.read_fields(c).cpu().numpy().astype(np.float64)
            ref = o.read_field(c)
            assert g.shape == ref.shape
            d = np.abs(g - ref).max()
            err[c] = max(err[c], d / scale if scale > 0 else d)
    rep = {"field_err": err, "emax": emax, "hmax": hmax}
    if len(w.get("freqs", [])) and w.get("ports"):
        dv = di = 0.0
        vs, is_ = [], []
        for p in range(len(w["ports"])):
            Vo, Io = o.read_port_dft(p)
            Vg, Ig = s.read_port_dft(p)
            vs.append((Vo, Vg))
            is_.append((Io, Ig))
        vmax = max(np.abs(v[0]).max() for v in vs)
        imax = max(np.abs(i[0]).max() for i in is_)
        for (Vo, Vg), (Io, Ig) in zip(vs, is_):
            dv = max(dv, np.abs(Vo - Vg).max() / vmax if vmax > 0 else 0.0)
            di = max(di, np.abs(Io - Ig).max() / imax if imax > 0 else 0.0)
        rep["dft_err"] = (dv, di)
    return o, s, rep


def assert_fields(rep, prec, tol=None):
    t = tol or TOL[prec]
    assert rep["emax"] > 0 and rep["hmax"] > 0, "nothing propagated: the test would be vacuous"
    assert rep["field_err"].max() <= t, f"field error {rep['field_err']} > {t}"
