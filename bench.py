"""bench.py -- throughput of the Yee FDTD hot path on config C3 (BASELINE.json: "Mcell-updates/s per Yee E+H step").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload c3|c3s|c0|c1|c2|c4|x3|w600]

One "step" is one full leapfrog step of the whole hot path (psi_H, H, psi_E, E, walls, source,
probes, running DFT) over the whole grid.  One cell-update = all six components of one cell advanced one step (R27);
N counts the CPML cells.  Prints ONE JSON line (rank 0).

  value         N_cells * K * n_gpus / t   with inputs resident in HBM, t from CUDA events around fdtd_step(K) on the
                solver's stream (barrier + synchronize on both sides, max over ranks)
  e2e           the same job through the C ABI with HOST buffers inside the timed region: material index + table
                host->device (fdtd_set_materials_indexed), fdtd_reset, K steps, every port's DFT device->host
  roofline      dominant kernel: algorithmic bytes per launch / its average duration from CUDA events
                (fdtd_profile_step) vs MEASURED_PEAKS.json hbm_gbs
  fused_step    c3 only, when fdtd_commit selected two steps per pass: the one-step fused E+H kernel on the same workload and
                step count, with its own roofline object (north_star's 70 % target is stated for that kernel's byte model)
  sustained     BASELINE.json's "2000 steps timed" on C3, with its own clock samples, whatever --steps says (c3 only;
                --sustained-steps 0 switches it off)
  cpu_baseline  the fp64 oracle, as it stands, on the host cores (all cores, and one thread), on the z-cropped
                1536x768x96 grid of the same generator (SURVEY 8(d) "Oracle timing"; full C3 needs ~150 GB of host
                arrays in fp64), rank 0, N=1
  --impl reference   times the oracle instead (there is no installable reference implementation: /root/reference holds
                a paper only); rank 0 alone works.

Multi-GPU.  north_star: one GPU, no sharding => the default mode is "replicas": every rank runs an
independent replica of the workload on its own GPU, no data-path collective; torch.distributed is used for the barrier
and the max of the times only.  `--mode sharded` is the z-slab decomposition of SURVEY 8(f) f4 (Table I:
weak scaling at 600^3 cells per GPU): one slab per rank, halo planes pushed into the neighbour's memory by the kernels.
With --gpus N > 1 and no WORLD_SIZE in the environment bench.py starts the N ranks itself (torchrun, 127.0.0.1) and the
line still comes from rank 0 with "n_gpus": N.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Mcell-updates/s per Yee E+H step"
UNIT = "Mcell-updates/s"


def csrc_hash():
    """sha256 (first 16 hex digits) over the kernel sources, in name order: ties an ncu capture to the build it was taken from."""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2208_04371_b200", "csrc", "*"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(workload_name, kernel, dtype, kz):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch from the `ncu --set full` capture recorded in
    profiles/traffic.json for exactly this (workload, kernel, dtype, kz, kernel-source hash); (None, why) otherwise."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(path):
        return None, "no profiles/traffic.json"
    sha = csrc_hash()
    near = None
    for e in json.load(open(path))["captures"]:
        if (e["workload"], e["kernel"], e["dtype"]) == (workload_name, kernel, dtype):
            if e["kz"] == kz and e["csrc_sha16"] == sha:
                return float(e["dram_bytes"]), e["source"]
            near = e
    if near is not None:
        return None, (f"capture in profiles/traffic.json is for kz={near['kz']}, csrc {near['csrc_sha16']} "
                      f"({near['dram_bytes'] / 1e9:.2f} GB); this run: kz={kz}, csrc {sha}")
    return None, "no capture of this workload / kernel in profiles/traffic.json"


def workload(name, steps):
    import workloads as W
    if name == "c3":
        return W.throughput_c3(steps=steps)
    if name == "c3s":  # 1/4-scale C3 for quick checks of this script (not a bench line)
        return W.throughput_c3(div=4, steps=steps, npml=16)
    if name == "c2":
        return W.interconnect_c2(steps=steps)
    if name == "c4":
        return W.interconnect_c4(steps=steps)
    if name == "c0":
        return W.cavity_c0(steps=steps)
    if name == "c1":
        return W.microstrip_c1(steps=steps)
    if name == "w600":  # the paper's per-GPU load of its weak-scaling study (Table I): 600^3 cells, C3's generator
        return W.weak_scaling_600(n_slabs=1, steps=steps)
    if name == "x3":  # the paper's CMOS-line grid shape, 200x120x800 cells of (20, 50, 5) nm
        return W.cmos_line_x3(steps=steps)
    raise SystemExit(f"unknown workload {name}")


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# --------------------------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks" line)
# --------------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, device_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        self.idx = device_index

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}", "--format=csv,noheader",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, reasons, power = [], [], set(), []
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1].split()[0]))
                smax.append(float(c[2].split()[0]))
                power.append(float(c[3].split()[0]))
            except ValueError:
                continue
            for n, v in zip(self.NAMES, c[5:9]):
                if v == "Active":
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": float(max(power))}


# --------------------------------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference): bounded sample of the same workload
# --------------------------------------------------------------------------------------------------------------------
# z-cropped C3 first (full-length rows and planes, 96 of the 768 planes); the smaller crops are fall-backs for
# hosts without the ~30 GB the fp64 oracle needs for it, and for the --impl reference arm's wall-clock bound
CPU_SAMPLE_LADDER = [(1536, 768, 96), (512, 384, 192), (384, 256, 160), (256, 192, 128), (192, 128, 96), (128, 96, 80)]
ORACLE_BYTES_PER_CELL = 8 * (6 + 9 + 6) + 8 * 6 + 2      # fields, coefficients, eps/sigma, the gather's temporaries, index


def _host_mem_available():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable:"):
                return int(line.split()[1]) * 1024
    except OSError:
        pass
    return 0


def _fits_host(shape):
    need = shape[0] * shape[1] * shape[2] * ORACLE_BYTES_PER_CELL
    avail = _host_mem_available()
    return avail == 0 or need * 1.3 < avail


def _oracle_on(shape):
    import workloads as W
    from oracle.yee import YeeOracle
    nb = max(1, int(4096 * (shape[0] * shape[1] * shape[2]) / (1536 * 768 * 768)))   # same block density as C3
    w = W.throughput_c3(shape=shape, steps=1, nblocks=nb)
    return YeeOracle.from_workload(w), w["nx"] * w["ny"] * w["nz"]


def _describe(shape, steps):
    return (f"fp64 oracle (g++ -O2 -fopenmp), C3 generator on {shape[0]}x{shape[1]}x{shape[2]} cells"
            f"{' (C3 cropped in z)' if shape[:2] == (1536, 768) else ' (bounded crop of C3)'}, 64-entry indexed materials, "
            f"16-cell six-face CPML, 4 ports, 128-frequency DFT, {steps} steps")


def oracle_sample(budget_s=15.0, steps=None, warmup=1, wall_s=150.0, one_thread=False):
    """Time the fp64 oracle as it stands on a bounded sample of C3.  With steps=None the step count fills budget_s on
    the largest crop the host holds; with steps given (the --impl reference arm) the crop is the largest of
    CPU_SAMPLE_LADDER whose steps+warmup steps are expected to fit in wall_s.
    Returns dict(value Mcell/s, s_per_step, steps, cores, sample, shape[, one_thread: {value, steps}])."""
    from oracle import yee
    ladder = [sh for sh in CPU_SAMPLE_LADDER if _fits_host(sh)] or CPU_SAMPLE_LADDER[-1:]
    shape = ladder[0]
    if steps is not None:
        o, n = _oracle_on(CPU_SAMPLE_LADDER[-1])
        o.step(1)
        t = time.perf_counter()
        o.step(2)
        rate = 2 * n / (time.perf_counter() - t)            # cells/s estimate
        del o
        for shape in ladder:
            if shape[0] * shape[1] * shape[2] * (steps + warmup) / rate <= wall_s:
                break
    o, n = _oracle_on(shape)
    cores = yee.num_threads()
    t = time.perf_counter()
    o.step(max(1, warmup))
    t1 = (time.perf_counter() - t) / max(1, warmup)
    if steps is None:
        steps = int(min(200, max(2, budget_s / t1)))
    t = time.perf_counter()
    o.step(steps)
    el = time.perf_counter() - t
    out = {"value": n * steps / el / 1e6, "s_per_step": el / steps, "steps": steps, "cores": cores,
           "sample": _describe(shape, steps), "shape": shape}
    if one_thread:
        n1 = int(max(1, min(steps, round(0.5 * budget_s / (el / steps * cores)))))   # about half the budget again
        yee.set_num_threads(1)
        try:
            t = time.perf_counter()
            o.step(n1)
            e1 = time.perf_counter() - t
        finally:
            yee.set_num_threads(cores)
        out["one_thread"] = {"value": n * n1 / e1 / 1e6, "unit": UNIT, "cores": 1, "steps": n1}
    return out


def run_reference(args, rank):
    if rank != 0:
        return
    # each "step" of this arm = one oracle step on the bounded crop; K steps after W warm-up steps
    r = oracle_sample(steps=args.steps, warmup=args.warmup)
    v, sps, k, cores, desc, shape = r["value"], r["s_per_step"], r["steps"], r["cores"], r["sample"], r["shape"]
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": k,
            "warmup": args.warmup, "ms_per_step": sps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "c3 (bounded sample, CPU oracle)", "grid": list(shape)},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
            "note": "no installable reference exists (/root/reference is a paper); this arm is the CPU oracle"}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------------------------
# algorithmic bytes per cell-update of the dominant kernel
# --------------------------------------------------------------------------------------------------------------------
def algorithmic_bytes(w, impl, kernel):
    """Bytes one launch of `kernel` must move, from the per-cell figures of SURVEY 8(d) / DESIGN.md:
    field words read and written once + the material operand + psi read+write on the slab cells."""
    n = w["nx"] * w["ny"] * w["nz"]
    es = 4 if w["precision"] == 32 else 8
    full = w["materials"]["mode"] == "full"
    mu = w["materials"].get("mu_r") is not None
    lo_hi = w["pml"]
    dims = (w["nx"], w["ny"], w["nz"])
    slab = sum((lo_hi[2 * a] + lo_hi[2 * a + 1]) * n // dims[a] for a in range(3))   # slab cells summed over axes
    psi_half = 2 * 2 * es * slab                     # two psi per slab-cell-axis per half step, read + write
    h_bytes = n * (6 * es + 3 * es + ((3 * es if full else 1) if mu else 0)) + psi_half
    e_bytes = n * (6 * es + 3 * es + (6 * es if full else 1)) + psi_half
    if impl == "fused":
        return n * (6 * es + 6 * es + (6 * es if full else 1) + ((3 * es if full else 0) if mu else 0)) + 2 * psi_half
    return h_bytes if kernel == "H" else e_bytes


# --------------------------------------------------------------------------------------------------------------------
# replicas: every rank runs the same workload on its own GPU; the job time is the max over ranks
# --------------------------------------------------------------------------------------------------------------------
def max_over_ranks(seconds, world, device):
    """The slowest rank's time (torch.distributed MAX all-reduce when world > 1; works with gloo on CPU tensors)."""
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(n_cells, steps, world, seconds):
    """Whole-job Mcell-updates/s: every rank advanced n_cells cells by `steps` steps in `seconds` (max over ranks)."""
    return n_cells * steps * world / seconds / 1e6


# --------------------------------------------------------------------------------------------------------------------
# the other configurations of BASELINE.json (and the paper's production grid shape) as short legs of the default run
# --------------------------------------------------------------------------------------------------------------------
OTHER_LEGS = (("c4", 150, 5), ("c2", 2000, 20), ("x3", 2000, 20), ("c1", 20000, 200), ("c0", 20000, 200))


def other_leg(name, K, Wm, dev, local_rank):
    """One short device-resident leg (W warm-up steps, K timed steps, CUDA events on the solver's stream, clocks sampled) of
    another workload: what fdtd_commit selects for it, its step time, and its own roofline object.  Grids that live in L2 (C0,
    C1) are launch- / barrier-bound, not bandwidth-bound: they report steps per second instead of a fraction."""
    import torch

    from paper_2208_04371_b200 import Solver
    t0 = time.perf_counter()
    w = workload(name, K)
    gen_s = time.perf_counter() - t0
    n_cells = w["nx"] * w["ny"] * w["nz"]
    s = Solver.from_workload(w, device=str(dev))
    s.step(Wm)
    torch.cuda.synchronize(dev)
    ck = ClockSampler(local_rank)
    ck.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.launch_count
    e0.record(s.stream)
    s.step(K)
    e1.record(s.stream)
    torch.cuda.synchronize(dev)
    clocks = ck.stop()
    t_s = e0.elapsed_time(e1) * 1e-3
    es = 4 if w["precision"] == 32 else 8
    leg = {"grid": [w["nx"], w["ny"], w["nz"]], "dtype": "f32" if es == 4 else "f64", "materials": w["materials"]["mode"],
           "steps": K, "warmup": Wm, "ms_per_step": t_s / K * 1e3, "value": n_cells * K / t_s / 1e6, "unit": UNIT,
           "step_impl": s.impl_name, "fused_kz": s.fused_kz, "fused_tile": s.fused_tile, "commit_s": s.commit_s,
           "generator_s": gen_s, "gpu_launches": s.launch_count - l0, "clocks": clocks}
    if s.impl_name == "persistent" or n_cells * 12 * es <= 100e6:
        leg["roofline"] = {"bound": "launch/barrier", "note": "grid and coefficients live in L2 (126 MB): no HBM roofline applies",
                           "steps_per_s": K / t_s, "us_per_step": t_s / K * 1e6}
    else:
        leg["roofline"], _ = kernel_roofline(s, w, K, t_s, name)
    s.destroy()
    del s
    torch.cuda.empty_cache()
    return leg


def kernel_roofline(s, w, K, t_s, workload_name):
    """The roofline object of one handle: per-kernel durations from fdtd_profile_step (CUDA events between the kernels, on the
    solver's stream), algorithmic bytes of the dominant kernel from the per-cell figures of DESIGN.md, the measured copy peak.
    Returns (roofline, bytes one step must move under the scheme in use)."""
    n_cells = w["nx"] * w["ny"] * w["nz"]
    ms = s.profile_step(max(3, min(20, K)))
    impl = s.impl_name
    es = 4 if w["precision"] == 32 else 8
    peak, peak_src = measured_peak()
    extra = {}
    if impl == "two_step":
        # the dominant kernel advances its box TWO steps per launch: every field of the box read once and written once (+1 B
        # index) per two cell-updates; profile_step's figures are per STEP, a launch lasts two of them.  The shell around the
        # box (CPML layers, port planes) is advanced step by step by the two-pass kernels on region grids (ms[1]).
        b = s.two_step_box
        box_cells = (b[1] - b[0]) * (b[3] - b[2]) * (b[5] - b[4])
        full = w["materials"]["mode"] == "full"
        kname, kms = "k_step2", 2.0 * ms[0]
        ab = box_cells * (12 * es + (6 * es if full else 1))
        shell_cells = n_cells - box_cells
        # what one STEP must move under this scheme: half a box pass + the shell's two-pass traffic (73 B fp32 indexed + psi)
        step_bytes = ab / 2 + (algorithmic_bytes(w, "two_pass", "H") + algorithmic_bytes(w, "two_pass", "E")) * shell_cells / n_cells
        one_step_model = algorithmic_bytes(w, "fused", "H")      # the 49 B + psi model of the one-step fused kernel, for comparison
        extra = {"box": b, "box_cells": box_cells, "shell_cells": shell_cells, "shell_ms_per_step": ms[1],
                 "bytes_per_cell_update_box": ab / 2 / box_cells,
                 "one_step_byte_model": {"bytes_per_cell_update": one_step_model / n_cells,
                                         "equivalent_gbs": one_step_model * K / t_s / 1e9,
                                         "equivalent_frac": one_step_model * K / t_s / 1e9 / peak,
                                         "note": "throughput expressed in the one-step fused kernel's byte model (49 B + psi per "
                                                 "cell-update): may exceed 1 because two steps per pass move fewer bytes"}}
    elif impl == "fused":
        kname, kms = "k_step_fused", ms[0]
        ab = algorithmic_bytes(w, impl, "H")
        step_bytes = ab
    else:
        kname, kms = ("k_update_E", ms[1]) if ms[1] >= ms[0] else ("k_update_H", ms[0])
        ab = algorithmic_bytes(w, impl, "E" if kname == "k_update_E" else "H")
        step_bytes = algorithmic_bytes(w, impl, "H") + algorithmic_bytes(w, impl, "E")
    achieved = ab / (kms * 1e-3) / 1e9
    # DRAM bytes of one launch from the committed `ncu --set full` capture of this workload and kernel (profiles/), else null
    traffic, traffic_src = ncu_traffic(workload_name, kname, "f32" if w["precision"] == 32 else "f64", s.fused_kz)
    roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": ab, "kernel_ms": kms,
                "kernel_ms_all": {"H_or_fused_or_box": ms[0], "E_or_shell": ms[1], "source": ms[2], "probe_dft": ms[3]},
                "bytes_per_cell_update_step": step_bytes / n_cells,
                "step_achieved_gbs": step_bytes * K / t_s / 1e9, "frac_of_8000": step_bytes * K / t_s / 1e9 / 8000.0}
    roofline.update(extra)
    return roofline, step_bytes


# --------------------------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------------------------
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist

    from paper_2208_04371_b200 import FDTD_OPT_FUSED_KZ, FDTD_OPT_FUSED_TILE, FDTD_OPT_STEP_IMPL, Solver, binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    K, Wm = args.steps, args.warmup
    w = workload(args.workload, K)
    n_cells = w["nx"] * w["ny"] * w["nz"]
    opts = {}
    if args.step_impl:
        opts[FDTD_OPT_STEP_IMPL] = args.step_impl
    if args.fused_kz:
        opts[FDTD_OPT_FUSED_KZ] = args.fused_kz
    if args.fused_tile:
        opts[FDTD_OPT_FUSED_TILE] = args.fused_tile
    s = Solver.from_workload(w, options=opts, device=str(dev))
    torch.cuda.synchronize(dev)

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps -------------------------------------
    s.step(Wm)
    barrier()
    clocks = ClockSampler(local_rank)
    clocks.start()
    l0 = s.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(s.stream)
    s.step(K)
    e1.record(s.stream)
    barrier()
    ck = clocks.stop()
    launches = s.launch_count - l0
    t_s = max_over_ranks(e0.elapsed_time(e1) * 1e-3, world, dev)
    value = job_throughput(n_cells, K, world, t_s)

    # ---- per-kernel durations (CUDA events between the kernels, on the solver's stream) ------------------------------
    impl = s.impl_name
    peak, peak_src = measured_peak()
    roofline, step_bytes = kernel_roofline(s, w, K, t_s, args.workload)

    # ---- sustained: BASELINE.json's "2000 steps timed" on C3, own clock samples ---------------------------------------
    sustained = None
    if args.workload == "c3" and args.sustained_steps > 0:
        barrier()
        ck2 = ClockSampler(local_rank)
        ck2.start()
        e0.record(s.stream)
        s.step(args.sustained_steps)
        e1.record(s.stream)
        barrier()
        c2 = ck2.stop()
        ts = max_over_ranks(e0.elapsed_time(e1) * 1e-3, world, dev)
        sustained = {"steps": args.sustained_steps, "ms_per_step": ts / args.sustained_steps * 1e3,
                     "value": job_throughput(n_cells, args.sustained_steps, world, ts), "unit": UNIT, "clocks": c2,
                     "step_achieved_gbs": step_bytes * args.sustained_steps / ts / 1e9,
                     "frac_of_peak": step_bytes * args.sustained_steps / ts / 1e9 / peak}

    # ---- end to end through the C ABI with host buffers ---------------------------------------------------------------
    m = w["materials"]
    e2e = None
    if m["mode"] == "indexed":
        idx_host = torch.from_numpy(np.ascontiguousarray(m["idx"], dtype=np.uint8)).pin_memory()
        nports, nf = len(w["ports"]), len(w["freqs"])
        barrier()
        t0 = time.perf_counter()
        s.set_materials_indexed(idx_host, m["eps_r"], m["sigma"], m.get("mu_r"))
        s.reset()
        s.step(K)
        out = [s.read_port_dft(p) for p in range(nports)]          # device -> host, synchronises
        torch.cuda.synchronize(dev)
        te = max_over_ranks(time.perf_counter() - t0, world, dev)
        h2d = idx_host.numel() + 12 * 256 * (4 if w["precision"] == 32 else 8)
        d2h = nports * nf * 2 * 2 * 8
        assert all(np.isfinite(v).all() and np.isfinite(i).all() for v, i in out)
        e2e = {"value": job_throughput(n_cells, K, world, te), "unit": UNIT,
               "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
               "what": "fdtd_set_materials_indexed(pinned host idx) + fdtd_reset + fdtd_step(K) + fdtd_read_port_dft x ports"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": t_s / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if w["precision"] == 32 else "f64", "data": "synthetic",
            "config": {"workload": args.workload, "grid": [w["nx"], w["ny"], w["nz"]], "cells": n_cells,
                       "materials": m["mode"], "cpml_cells": w["pml"], "ports": len(w["ports"]), "dft_freqs": len(w["freqs"]),
                       "step_impl": impl, "commit_s": s.commit_s, "fused_kz": s.fused_kz, "fused_tile": s.fused_tile, "l2": "inputs larger than L2 (no flush needed)" if n_cells * 24 > 2.6e8 else
                       "grid fits in L2: launch-bound case, not a roofline case",
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "library": os.path.basename(binding.library_path())},
            "clocks": ck, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "sustained": sustained}
    s.destroy()
    del s
    torch.cuda.empty_cache()
    # ---- the one-step fused kernel beside a two-step headline (c3): north_star's ">= 70 % of HBM bandwidth for the fused E+H step" is
    # a statement about THAT kernel's 49 B + psi per cell-update; the same K steps, timed the same way, on a second handle
    if impl == "two_step" and args.workload == "c3" and not args.step_impl and not args.no_fused_leg:
        s1 = Solver.from_workload(w, options={FDTD_OPT_STEP_IMPL: 2}, device=str(dev))
        s1.step(Wm)
        barrier()
        e0.record(s1.stream)
        s1.step(K)
        e1.record(s1.stream)
        barrier()
        t1 = max_over_ranks(e0.elapsed_time(e1) * 1e-3, world, dev)
        m1 = s1.profile_step(max(3, min(20, K)))
        ab1 = algorithmic_bytes(w, "fused", "H")
        tr1, tr1_src = ncu_traffic(args.workload, "k_step_fused", "f32" if w["precision"] == 32 else "f64", s1.fused_kz)
        line["fused_step"] = {"what": "FDTD_OPT_STEP_IMPL = 2 (one step per pass), same workload, same K steps",
                              "ms_per_step": t1 / K * 1e3, "value": job_throughput(n_cells, K, world, t1), "unit": UNIT,
                              "fused_kz": s1.fused_kz, "fused_tile": s1.fused_tile,
                              "roofline": {"bound": "hbm", "kernel": "k_step_fused", "achieved": ab1 / (m1[0] * 1e-3) / 1e9, "peak": peak,
                                           "unit": "GB/s", "frac": ab1 / (m1[0] * 1e-3) / 1e9 / peak, "traffic": tr1,
                                           "traffic_source": tr1_src, "algorithmic_bytes_per_launch": ab1, "kernel_ms": m1[0],
                                           "frac_of_8000": ab1 / (m1[0] * 1e-3) / 1e9 / 8000.0}}
        s1.destroy()
        del s1
        torch.cuda.empty_cache()
    if rank == 0 and world == 1 and args.workload == "c3" and not args.no_others:
        line["others"] = {name: other_leg(name, k, wm, dev, local_rank) for name, k, wm in OTHER_LEGS}
    if rank == 0 and world == 1 and not args.no_cpu:
        r = oracle_sample(budget_s=args.cpu_budget, one_thread=True)
        line["cpu_baseline"] = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
                                "one_thread": r.get("one_thread")}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------------------------------
# --mode sharded: z-slab decomposition, weak scaling at 600^3 cells per GPU (Table I)
# --------------------------------------------------------------------------------------------------------------------
def run_sharded(args, rank, world, local_rank):
    """One 600^3 slab per rank of a 600 x 600 x 600N grid; the slabs push their boundary planes into each other's halo from
    the kernels (paper_2208_04371_b200/sharded.py).  With ONE rank and --slabs S the rank's grid is cut into S slabs on its
    own GPU instead (they share a stream): that measures what the protocol itself costs, not a scaling point."""
    import torch
    import torch.distributed as dist

    import workloads as W
    from paper_2208_04371_b200 import binding
    from paper_2208_04371_b200.sharded import DistributedSlab, ShardedSolver

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    K, Wm = args.steps, args.warmup
    on_one_gpu = world == 1
    n_slabs = world if world > 1 else max(1, args.slabs)
    per_gpu = 1 if world > 1 else n_slabs                      # slabs that share this rank's GPU
    edge = args.edge
    # weak scaling: edge^3 cells per GPU.  One rank with --slabs S keeps ONE GPU's load (edge^2 x edge planes) and cuts it.
    w = W.weak_scaling_600(n_slabs=world, steps=K, edge=edge)
    n_cells = w["nx"] * w["ny"] * w["nz"]
    if on_one_gpu:
        sim = ShardedSolver(w, [str(dev)] * n_slabs)
        stream = sim.solvers[0].stream
        first = sim.solvers[0]
    else:
        sim = DistributedSlab(w, str(dev), transport="peer")
        stream = sim.solver.stream
        first = sim.solver
    torch.cuda.synchronize(dev)
    sim.step(Wm)
    barrier()
    clocks = ClockSampler(local_rank)
    clocks.start()
    l0 = sim.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    sim.step(K)
    e1.record(stream)
    barrier()
    ck = clocks.stop()
    launches = sim.launch_count - l0
    t_s = max_over_ranks(e0.elapsed_time(e1) * 1e-3, world, dev)
    value = n_cells * K / t_s / 1e6
    ab = algorithmic_bytes(dict(w, nz=w["nz"] // world, pml=w["pml"][:4] + [w["pml"][4] if world == 1 else 0, w["pml"][5] if world == 1 else 0]),
                           "fused", "H")
    peak, peak_src = measured_peak()
    # end to end: every slab's material slice from pinned host memory, reset, K steps, the port DFTs back to the host
    barrier()
    t0 = time.perf_counter()
    h2d = sim.upload_materials(pinned=True) if on_one_gpu else sim.upload_materials(w, pinned=True)
    sim.reset()
    sim.step(K)
    out = [sim.read_port_dft(p) for p in range(len(w["ports"]))]
    torch.cuda.synchronize(dev)
    te = max_over_ranks(time.perf_counter() - t0, world, dev)
    assert all(np.isfinite(v).all() and np.isfinite(i).all() for v, i in out)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": t_s / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": w["name"], "grid": [w["nx"], w["ny"], w["nz"]], "cells": n_cells,
                       "cells_per_gpu": n_cells // world, "materials": "indexed", "cpml_cells": w["pml"], "ports": len(w["ports"]),
                       "dft_freqs": len(w["freqs"]), "step_impl": first.impl_name, "fused_kz": first.fused_kz,
                       "parallelism": (f"z-slabs x{world}, one per GPU, halo planes stored into the neighbour by the kernels (NVLink peer stores)"
                                       if world > 1 else f"1 GPU, its grid cut into {per_gpu} z slab(s) on the same device (protocol cost only)"),
                       "l2": "inputs larger than L2 (no flush needed)", "library": os.path.basename(binding.library_path())},
            "clocks": ck,
            "e2e": {"value": n_cells * K / te / 1e6, "unit": UNIT, "h2d_bytes_per_step": h2d / K,
                    "d2h_bytes_per_step": len(w["ports"]) * len(w["freqs"]) * 32 / K,
                    "what": "per slab: fdtd_set_materials_indexed(pinned host slice) + fdtd_reset; K steps; fdtd_read_port_dft x ports"},
            "gpu_launches": launches,
            "roofline": {"bound": "hbm", "kernel": "k_step_fused (one slab's step incl. hand-over kernels)", "achieved": ab / (t_s / K) / 1e9,
                         "peak": peak, "unit": "GB/s", "frac": ab / (t_s / K) / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": ab}}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def spawn_ranks(n):
    """`python bench.py --gpus N` without a launcher: start the N ranks under torchrun (one process per GPU, rendezvous on
    127.0.0.1) with this command line; rank 0 of that job prints the line."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3")
    ap.add_argument("--step-impl", type=int, default=0, help="FDTD_OPT_STEP_IMPL: 0 auto, 1 two-pass, 2 fused, 3 persistent, 4 two steps per pass")
    ap.add_argument("--fused-kz", type=int, default=0, help="FDTD_OPT_FUSED_KZ: planes per z chunk (0 = measured at commit)")
    ap.add_argument("--fused-tile", type=int, default=0, help="FDTD_OPT_FUSED_TILE: 0 measured at commit, 1 = 14-row tiles, 2 = 6-row tiles")
    ap.add_argument("--no-fused-leg", action="store_true", help="c3, two steps per pass selected: skip the one-step fused kernel's leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-others", action="store_true", help="c3: skip the short legs of the other configurations (c4, c2, x3, c1, c0)")
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--sustained-steps", type=int, default=2000,
                    help="steps of the sustained leg on c3 (BASELINE.json: '2000 steps timed'); 0 = off")
    ap.add_argument("--mode", default="replicas", choices=["replicas", "sharded"],
                    help="multi-GPU: independent replicas (default) or one z slab of a (600 x 600 x 600 N) grid per rank")
    ap.add_argument("--slabs", type=int, default=0,
                    help="--mode sharded on ONE rank: cut the rank's grid into this many slabs on its GPU (protocol cost)")
    ap.add_argument("--edge", type=int, default=600, help="--mode sharded: cells per GPU = edge^3 (the paper's Table I: 600)")
    args = ap.parse_args()
    args.warmup = max(3, args.warmup)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args.gpus)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.mode == "sharded":
        run_sharded(args, rank, world, local_rank)
        return
    run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
