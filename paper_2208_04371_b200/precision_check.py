"""fp32 against fp64 time stepping at a config's FULL step count, both on the GPU (R14).

    python -m paper_2208_04371_b200.precision_check [--steps 200000]

The CPU oracle cannot reach C2's 200 000 steps (hours); the library's fp64 mode, which matches the oracle to 1e-11 on
every rung the oracle does reach, stands in for it here to answer one question: does fp32 time stepping itself keep S*
within north_star's 1e-3 over a full-length run (SURVEY G31 extrapolated a risk of 2.5e-3 for S*_11)?  Inc and tot runs of
config C2 in both precisions, S* column by Eq. 1-2, printed differences.  A measurement, not a parity test.
"""
import argparse
import os
import sys
import time

import numpy as np

from . import FDTD_F32, FDTD_F64, Solver, sparams


def main():
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import torch
    import workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=200000)
    a = ap.parse_args()
    res = {}
    for prec in (FDTD_F32, FDTD_F64):
        for run in ("inc", "tot"):
            w = W.interconnect_c2(run=run, steps=a.steps)
            s = Solver.from_workload(w, precision=prec)
            t = time.time()
            s.step(a.steps)
            torch.cuda.synchronize()
            el = time.time() - t
            V, I = zip(*[s.read_port_dft(p) for p in range(len(w["ports"]))])
            res[(prec, run)] = (np.array(V), np.array(I))
            print(f"fp{prec} {run}: {s.impl_name}, {el:.1f} s, {el / a.steps * 1e3:.4f} ms/step, finite={np.isfinite(np.array(V)).all()}", flush=True)
            s.destroy()
    S = {p: sparams.s_star_column(0, res[(p, "inc")][0], res[(p, "inc")][1], res[(p, "tot")][0]) for p in (FDTD_F32, FDTD_F64)}
    d = np.abs(S[FDTD_F32] - S[FDTD_F64])
    print(f"max |dS*_11| = {d[0].max():.3e}   max |dS*_21| = {d[1].max():.3e}   (north_star: 1e-3)")
    v32, v64 = res[(FDTD_F32, "tot")][0], res[(FDTD_F64, "tot")][0]
    print(f"raw port DFT, fp32 against fp64, relative to the band maximum: {np.abs(v32 - v64).max() / np.abs(v64).max():.3e}")


if __name__ == "__main__":
    main()
