"""Seeded random sweep over shapes (around the tile, chunk and vector boundaries of the kernels), CPML thicknesses per
face, material encodings, permeability, precision, step implementation and chunk length: every case against the oracle.
(400 cases of the same generator were run once during round 1 without a failure; 48 stay in the suite.)"""
import numpy as np
import pytest

import workloads as W
from paper_2208_04371_b200 import FDTD_F32, FDTD_F64, FDTD_OPT_FUSED_KZ, FDTD_OPT_FUSED_TILE, FDTD_OPT_STEP_IMPL, FdtdError, Solver
from tests.parity_util import TOL, run_pair

pytestmark = pytest.mark.gpu


def _cases(seed, n):
    r = np.random.default_rng(seed)
    for case in range(n):
        nx = int(r.choice([r.integers(18, 60), r.integers(120, 140), r.integers(250, 262), 128, 256, 64]))
        ny = int(r.choice([r.integers(10, 20), r.integers(26, 31), 14, 28, 42, r.integers(40, 60)]))
        nz = int(r.choice([r.integers(10, 30), r.integers(30, 70), 24, 36, 48]))
        pml = [int(r.choice([0, 0, r.integers(2, 7), 4, 8])) for _ in range(6)]
        for a, n_ in enumerate((nx, ny, nz)):
            while pml[2 * a] + pml[2 * a + 1] > n_ - 6:
                pml[2 * a] //= 2
                pml[2 * a + 1] //= 2
        yield dict(case=case, nx=nx, ny=ny, nz=nz, pml=tuple(pml), indexed=bool(r.integers(0, 2)), mu=bool(r.integers(0, 2)),
                   prec=int(r.choice([FDTD_F32, FDTD_F64])), impl=int(r.choice([1, 2, 3])), kz=int(r.choice([0, 3, 7, 12, 16])),
                   steps=int(r.integers(20, 70)))


@pytest.mark.parametrize("seed", [3, 5, 8])
def test_random_configurations_against_the_oracle(seed):
    for c in _cases(seed, 16):
        w = W.random_box(2000 + 100 * seed + c["case"], nx=c["nx"], ny=c["ny"], nz=c["nz"], pml=c["pml"], indexed=c["indexed"],
                         with_mu=c["mu"], precision=c["prec"], steps=c["steps"])
        opts = {FDTD_OPT_STEP_IMPL: c["impl"]}
        if c["impl"] == 2:
            opts[FDTD_OPT_FUSED_KZ] = c["kz"]
            opts[FDTD_OPT_FUSED_TILE] = 1 + (c["case"] + seed) % 2      # both tile shapes of the fused kernel
        o, s, rep = run_pair(w, c["steps"], precision=c["prec"], options=opts, checkpoints=[max(1, c["steps"] // 2), c["steps"]])
        assert rep["emax"] > 0, c
        assert rep["field_err"].max() <= TOL[c["prec"]], (c, rep["field_err"])
        assert max(rep["dft_err"]) <= (1e-4 if c["prec"] == FDTD_F32 else 1e-11), (c, rep["dft_err"])
        s.destroy()


def test_random_configurations_two_steps_per_pass():
    """The same kind of sweep for FDTD_OPT_STEP_IMPL = 4 on grids large enough to hold a box: shapes around the 120-cell
    owned tile width and the 8-row owned tile height, CPML on random faces, both material encodings, chunk lengths that do
    and do not divide the box, odd and even step counts.  Grids that leave no box are counted, not failed."""
    r = np.random.default_rng(44)
    ran = refused = 0
    for case in range(14):
        nx = int(r.choice([r.integers(110, 135), r.integers(236, 250), r.integers(300, 330), 128, 256]))
        ny = int(r.choice([r.integers(24, 34), r.integers(40, 60), 28, 36]))
        nz = int(r.choice([r.integers(20, 40), 24, 33, 48]))
        pml = tuple(int(r.choice([0, 0, r.integers(2, 7), 4])) for _ in range(6))
        prec = int(r.choice([FDTD_F32, FDTD_F64]))
        steps = int(r.integers(9, 40))
        w = W.random_box(4400 + case, nx=nx, ny=ny, nz=nz, pml=pml, indexed=bool(r.integers(0, 2)), with_mu=bool(r.integers(0, 2)),
                         precision=prec, steps=steps)
        opts = {FDTD_OPT_STEP_IMPL: 4, FDTD_OPT_FUSED_KZ: int(r.choice([0, 3, 7, 12, 16]))}
        try:
            Solver.from_workload(w, precision=prec, options=opts).destroy()
        except FdtdError as e:
            assert e.code == -1
            refused += 1
            continue
        o, s, rep = run_pair(w, steps, precision=prec, options=opts, checkpoints=[max(1, steps // 2), steps])
        assert s.impl_name == "two_step" and rep["emax"] > 0
        assert rep["field_err"].max() <= TOL[prec], (case, nx, ny, nz, pml, rep["field_err"])
        assert max(rep["dft_err"]) <= (1e-4 if prec == FDTD_F32 else 1e-11), (case, rep["dft_err"])
        s.destroy()
        ran += 1
    assert ran >= 8, (ran, refused)
