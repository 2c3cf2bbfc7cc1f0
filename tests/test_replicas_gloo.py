"""N > 1 is "replicas only": no data-path collective, only the barrier and the max-over-ranks of the step
time.  This covers that host-side logic of bench.py with world_size = 2 on the gloo backend (CPU)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local = 0.010 if rank == 0 else 0.025                     # rank 1 is the slow replica
    t = bench.max_over_ranks(local, world, torch.device("cpu"))
    dist.barrier()
    out[rank] = (t, bench.job_throughput(1000, 7, world, t))
    dist.destroy_process_group()


def test_replicas_time_is_max_over_ranks_and_value_is_whole_job():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    t, v = res[0]
    assert t == 0.025
    assert v == 1000 * 7 * 2 / 0.025 / 1e6


def test_single_rank_needs_no_process_group():
    assert bench.max_over_ranks(0.5, 1, torch.device("cpu")) == 0.5


def test_algorithmic_bytes_are_the_per_cell_figures_of_the_scope_table():
    """bench.py's roofline numerator: C3 in fp32 with a uint8 index -- 49 B per cell for the fused
    step, 36 / 37 B for the H / E pass, plus 16 B per slab-cell-axis and half step for psi; C4 in fp64 with full coefficient
    arrays -- 144 B fused, 72 / 120 B two-pass.  Checked on descriptors only (no arrays are generated)."""
    c3 = dict(nx=1536, ny=768, nz=768, precision=32, pml=[16] * 6, materials={"mode": "indexed", "mu_r": None})
    n = 1536 * 768 * 768
    slab = 32 * (768 * 768 + 1536 * 768 + 1536 * 768)
    assert slab == 94371840
    assert bench.algorithmic_bytes(c3, "fused", "H") == 49 * n + 32 * slab == 47412412416
    assert bench.algorithmic_bytes(c3, "two_pass", "H") == 36 * n + 16 * slab
    assert bench.algorithmic_bytes(c3, "two_pass", "E") == 37 * n + 16 * slab
    c4 = dict(nx=1024, ny=512, nz=256, precision=64, pml=[12, 12, 12, 12, 0, 12], materials={"mode": "full", "mu_r": None})
    n4 = 1024 * 512 * 256
    slab4 = 24 * 512 * 256 + 24 * 1024 * 256 + 12 * 1024 * 512
    assert bench.algorithmic_bytes(c4, "fused", "H") == 144 * n4 + 64 * slab4
    assert bench.algorithmic_bytes(c4, "two_pass", "H") == 72 * n4 + 32 * slab4
    assert bench.algorithmic_bytes(c4, "two_pass", "E") == 120 * n4 + 32 * slab4


def test_traffic_lookup_is_keyed_on_the_kernel_source_hash():
    """profiles/traffic.json entries are quoted only for the build they were captured on."""
    sha = bench.csrc_hash()
    t, src = bench.ncu_traffic("c3", "k_step2", "f32", 96)
    import json
    caps = json.load(open(os.path.join(bench.ROOT, "profiles", "traffic.json")))["captures"]
    mine = [e for e in caps if (e["workload"], e["kernel"], e["dtype"], e["kz"]) == ("c3", "k_step2", "f32", 96)]
    assert len(mine) == 1
    if mine[0]["csrc_sha16"] == sha:
        assert t == float(mine[0]["dram_bytes"])
    else:
        assert t is None and "csrc" in src
    assert bench.ncu_traffic("c3", "k_step2", "f32", 95)[0] is None          # another chunk length: no figure
    assert bench.ncu_traffic("nothing", "k_step2", "f32", 96)[0] is None
