"""Seeded random sweep over shapes (around the tile, chunk and vector boundaries of the kernels), CPML thicknesses per
face, material encodings, permeability, precision, step implementation and chunk length: every case against the oracle.
(400 cases of the same generator were run once during round 1 without a failure; 48 stay in the suite.)"""
import numpy as np
import pytest

import workloads as W
from paper_2208_04371_b200 import FDTD_F32, FDTD_F64, FDTD_OPT_FUSED_KZ, FDTD_OPT_STEP_IMPL
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
        o, s, rep = run_pair(w, c["steps"], precision=c["prec"], options=opts, checkpoints=[max(1, c["steps"] // 2), c["steps"]])
        assert rep["emax"] > 0, c
        assert rep["field_err"].max() <= TOL[c["prec"]], (c, rep["field_err"])
        assert max(rep["dft_err"]) <= (1e-4 if c["prec"] == FDTD_F32 else 1e-11), (c, rep["dft_err"])
        s.destroy()
