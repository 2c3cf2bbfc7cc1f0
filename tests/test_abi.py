"""The C-ABI library loads and exports every symbol include/fdtd.h declares; host-side argument checks (no GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2208_04371_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "fdtd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fdtd_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = declared_symbols()
    assert len(names) >= 20 and "fdtd_step" in names and "fdtd_read_port_dft" in names
    L = ctypes.CDLL(B._build.build())
    for n in names:
        assert hasattr(L, n), f"libfdtd_b200.so does not export {n}"
    assert sorted(B.SYMBOLS) == names, "binding.py and include/fdtd.h disagree on the symbol list"


def test_library_has_no_torch_or_oracle_dependency():
    import subprocess
    out = subprocess.run(["ldd", B._build.build()], capture_output=True, text=True).stdout
    assert "torch" not in out and "oracle" not in out and "libcudart" not in out  # static runtime, plain C ABI


def test_create_argument_checks():
    with pytest.raises(B.FdtdError) as e:
        B.fdtd_create(1, 8, 8, 1e-9, 1e-9, 1e-9, 1e-18)
    assert e.value.code == B.FDTD_EINVAL
    with pytest.raises(B.FdtdError) as e:
        B.fdtd_create(8, 8, 8, 1e-9, 1e-9, 1e-9, 1e-18, precision=16)
    assert e.value.code == B.FDTD_EINVAL
    # the CFL limit: dt <= 1/(c sqrt(1/dx^2 + 1/dy^2 + 1/dz^2))
    lim = 1.0 / (299792458.0 * np.sqrt(1 / 20e-9**2 + 1 / 50e-9**2 + 1 / 5e-9**2))
    h = B.fdtd_create(8, 8, 8, 20e-9, 50e-9, 5e-9, lim * (1 - 1e-12))
    B.fdtd_destroy(h)
    with pytest.raises(B.FdtdError) as e:
        B.fdtd_create(8, 8, 8, 20e-9, 50e-9, 5e-9, lim * (1 + 1e-9))
    assert e.value.code == B.FDTD_ECFL


def test_setup_checks_and_lifecycle_without_gpu():
    h = B.fdtd_create(16, 12, 10, 1e-9, 1e-9, 1e-9, 1e-18)
    try:
        with pytest.raises(B.FdtdError) as e:
            B.fdtd_set_boundary(h, [9, 8, 0, 0, 0, 0])
        assert e.value.code == B.FDTD_ERANGE
        with pytest.raises(B.FdtdError) as e:
            B.fdtd_set_boundary(h, [2] * 6, [3, 1, 0.5, 0, 0.8, 1])      # kappa_max < 1
        assert e.value.code == B.FDTD_EINVAL
        B.fdtd_set_boundary(h, [2, 2, 2, 2, 0, 2])
        small = B.fdtd_workspace_bytes(h)
        port = dict(has_source=1, sj0=4, sj1=6, sk0=0, sk1=3, waveform=1, amp=1.0, t0=3e-17, sigma=1e-17, f0=0.0,
                    ip=5, vj0=4, vj1=6, vk0=0, vk1=3, lj0=3, lj1=7, lk0=2, lk1=4)
        port["is"] = 4
        assert B.fdtd_add_port(h, port) == 0
        bad = dict(port, lj0=0)
        with pytest.raises(B.FdtdError) as e:
            B.fdtd_add_port(h, bad)
        assert e.value.code == B.FDTD_ERANGE
        bad = dict(port, vk1=11)
        with pytest.raises(B.FdtdError) as e:
            B.fdtd_add_port(h, bad)
        assert e.value.code == B.FDTD_ERANGE
        for wall in (dict(port, sj0=0), {**port, "is": 0}):      # E_z on i = 0 / j = 0 is a PEC wall sample (R1)
            with pytest.raises(B.FdtdError) as e:
                B.fdtd_add_port(h, wall)
            assert e.value.code == B.FDTD_ERANGE
        assert B.fdtd_device(h) == -1 and B.fdtd_graph_replays(h) == 0
        B.fdtd_set_dft(h, np.linspace(1e9, 5e11, 128))
        B.fdtd_set_material_mode(h, B.FDTD_MAT_FULL, True)
        assert B.fdtd_workspace_bytes(h) > small            # nine coefficient arrays instead of an index
        with pytest.raises(B.FdtdError) as e:
            B.fdtd_set_option(h, 99, 1)
        assert e.value.code == B.FDTD_EINVAL
        # everything that needs the device state is refused before commit
        with pytest.raises(B.FdtdError) as e:
            B.fdtd_step(h, 1)
        assert e.value.code == B.FDTD_ESTATE
        assert B.fdtd_step_count(h) == 0 and B.fdtd_impl_name(h) == ""
        import torch
        if not torch.cuda.is_available():
            # no CPU fallback: commit fails loudly without a CUDA device
            with pytest.raises(B.FdtdError) as e:
                B.fdtd_commit(h, torch.empty(1024, dtype=torch.uint8), 0)
            assert e.value.code == B.FDTD_ECUDA
            assert "no CPU fallback" in str(e.value)
    finally:
        B.fdtd_destroy(h)


def test_workspace_size_is_the_documented_layout():
    """fp32 indexed: padded field arrays + one padded byte array dominate; psi only on the slabs.
    At this size the step is the fused kernel: two field sets (ping-pong) and a second copy of the six psi_H families;
    forcing the two-pass step (FDTD_OPT_STEP_IMPL = 1) gives the single-set layout."""
    nx, ny, nz = 1536, 768, 768
    P = (nx + 1 + 31) // 32 * 32
    padded = P * (ny + 1) * (nz + 2)
    fam = 4 * (2 * 32 * ny * nz + 2 * P * 32 * nz + 2 * P * ny * 32)      # one family group: 2 psi arrays per axis
    for impl, nsets, ngroups in ((1, 1, 2), (0, 2, 3)):
        h = B.fdtd_create(nx, ny, nz, 5e-9, 5e-9, 5e-9, 9e-18)
        B.fdtd_set_boundary(h, [16] * 6)
        B.fdtd_set_option(h, B.FDTD_OPT_STEP_IMPL, impl)
        expect = nsets * 6 * 4 * padded + padded + ngroups * fam
        got = B.fdtd_workspace_bytes(h)
        B.fdtd_destroy(h)
        assert expect <= got <= expect * 1.01 + (1 << 20), (impl, expect, got)


def test_binding_refuses_material_arrays_of_the_wrong_type_or_size():
    """The C side sees bare pointers, so the binding checks element type, count and contiguity first (no GPU needed:
    the check runs before the library is called)."""
    n = 6 * 5 * 4
    ok = [np.ones(n, dtype=np.float32)] * 3
    for bad in ([np.ones(n, dtype=np.float64)] * 3, [np.ones(n - 1, dtype=np.float32)] * 3, [np.ones(n, dtype=np.int32)] * 3,
                ok[:2]):
        with pytest.raises(ValueError):
            B.fdtd_set_materials_full(None, bad, ok, n_cells=n, precision=B.FDTD_F32)
    with pytest.raises(ValueError):
        B.fdtd_set_materials_full(None, ok, [np.ones((n, 2), dtype=np.float32)[:, 0]] * 3, n_cells=n, precision=B.FDTD_F32)
