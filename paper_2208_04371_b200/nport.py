"""N-port S-parameter extraction: the paper's two-run protocol around the GPU time loop.

For every driving port j: an "inc" run on the uniform line (no reflections: V_inc, I_inc) and a "tot" run on the full
circuit with the same source (V_tot, V_tra); 2 N runs for an N x N matrix.  Then, host side, O(N^2 F):
    Z_r(y_j)  = F[V_inc(y_j)] / F[I_inc(y_j)]                          (Eq. 2)
    S*[:, j]  = Eq. 1 (sparams.s_star_column)
    S         = Eq. 5-6 renormalisation of S* to 50 ohm (sparams.renormalize)
    tau_ij    = Eq. 8 phase delay of S*_ij (sparams.phase_delay)
Orientation (R7, R31): the library's current loop is right-handed about +x and V = +int E_z dz, so a wave
travelling towards +x has Re(V/I) < 0.  Z_r is reported for a current that flows with the incident wave and a voltage of
the strip against the ground, Z_r = -d_j V/I with d_j = +1 for a port driven towards +x: Re Z_r > 0, which Eq. 5 needs.
Every run is an independent simulation (the replica unit of DESIGN.md 8): `devices` may list several GPUs, and the 2 N
runs are then dealt out to them, one worker thread per device (the library calls release the GIL; each handle carries its
own device and stream).
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from . import sparams
from .solver import Solver


def _run(w, steps, device, options):
    s = Solver.from_workload(w, options=options, device=device)
    s.step(steps)
    nports = len(w["ports"])
    V = np.empty((nports, len(w["freqs"])), dtype=np.complex128)
    I = np.empty_like(V)
    for p in range(nports):
        V[p], I[p] = s.read_port_dft(p)
    s.destroy()
    return V, I


def extract(workload_for_run, drive_port, steps=None, device="cuda:0", options=None, z_new=50.0, ports=None, devices=None):
    """workload_for_run(run) -> workload dict for run in ("inc", "tot") with one driving port (workloads/ generators);
    drive_port(w, j) -> (workload with port j driving, direction).  devices: GPUs to spread the runs over (default: the one
    `device`).  Returns a dict with S_star [N,N,F], Z_r [N,F], S [N,N,F] (on z_new ohm), tau [N,N,F] (Eq. 8; diagonal = nan)
    and freqs."""
    w_inc, w_tot = workload_for_run("inc"), workload_for_run("tot")
    n = len(w_inc["ports"])
    freqs = np.asarray(w_inc["freqs"], dtype=np.float64)
    steps = int(steps if steps is not None else w_inc["steps"])
    drive = list(range(n)) if ports is None else list(ports)
    devs = list(devices) if devices else [device]
    S_star = np.full((n, n, freqs.size), np.nan, dtype=np.complex128)
    Z_r = np.full((n, freqs.size), np.nan, dtype=np.complex128)
    # the independent runs, dealt round-robin to the devices; each device works through its share in order
    jobs = []
    direction = {}
    for j in drive:
        wi, direction[j] = drive_port(w_inc, j)
        wt, _ = drive_port(w_tot, j)
        jobs += [((j, "inc"), wi), ((j, "tot"), wt)]
    shares = [jobs[q::len(devs)] for q in range(len(devs))]

    def work(q):
        return [(key, _run(w, steps, devs[q], options)) for key, w in shares[q]]

    if len(devs) == 1:
        done = work(0)
    else:
        with ThreadPoolExecutor(max_workers=len(devs)) as pool:
            done = [r for part in pool.map(work, range(len(devs))) for r in part]
    res = dict(done)
    for j in drive:
        Vi, Ii = res[(j, "inc")]
        Vt, _ = res[(j, "tot")]
        S_star[:, j] = sparams.s_star_column(j, Vi, Ii, Vt)
        Z_r[j] = -direction[j] * Vi[j] / Ii[j]
    out = {"freqs": freqs, "S_star": S_star, "Z_r": Z_r}
    if len(drive) == n:
        out["S"] = sparams.renormalize(S_star, Z_r, z_new)
        tau = np.full((n, n, freqs.size), np.nan)
        for i in range(n):
            for j in range(n):
                if i != j:
                    tau[i, j] = sparams.phase_delay(S_star[i, j], freqs)
        out["tau"] = tau
    return out
