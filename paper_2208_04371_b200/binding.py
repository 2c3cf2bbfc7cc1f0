"""ctypes binding of include/fdtd.h -- argument marshalling only; every step of the method runs in the CUDA library.

Module-level functions carry the names of the C ABI (fdtd_create, fdtd_set_boundary, ..., fdtd_destroy) and take the
handle first.  `Solver` is a small convenience wrapper around them that owns the handle and the torch workspace.
PyTorch is used for exactly two things: the device workspace (`torch.empty(..., dtype=uint8, device="cuda")`) and the
current CUDA stream.  There is no CPU fallback: if the library cannot be built or loaded, importing fails loudly.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

FDTD_OK, FDTD_EINVAL, FDTD_ECFL, FDTD_ESTATE, FDTD_ENOMEM, FDTD_ECUDA, FDTD_ERANGE = 0, -1, -2, -3, -4, -5, -6
FDTD_F32, FDTD_F64 = 32, 64
FDTD_W_DGAUSS, FDTD_W_GAUSS, FDTD_W_GSINE = 0, 1, 2
FDTD_MAT_INDEXED, FDTD_MAT_FULL = 0, 1
FDTD_EX, FDTD_EY, FDTD_EZ, FDTD_HX, FDTD_HY, FDTD_HZ = range(6)
FDTD_OPT_STEP_IMPL, FDTD_OPT_USE_GRAPH, FDTD_OPT_GRAPH_UNROLL, FDTD_OPT_FUSED_KZ, FDTD_OPT_Z_SPIN, FDTD_OPT_FUSED_TILE = 1, 2, 3, 4, 5, 6
FDTD_OPT_TUNE_MEMO = 7

_ERRNAMES = {-1: "FDTD_EINVAL", -2: "FDTD_ECFL", -3: "FDTD_ESTATE", -4: "FDTD_ENOMEM", -5: "FDTD_ECUDA", -6: "FDTD_ERANGE"}


class fdtd_port(C.Structure):
    _fields_ = [("has_source", C.c_int),
                ("is_", C.c_int), ("sj0", C.c_int), ("sj1", C.c_int), ("sk0", C.c_int), ("sk1", C.c_int),
                ("waveform", C.c_int),
                ("amp", C.c_double), ("t0", C.c_double), ("sigma", C.c_double), ("f0", C.c_double),
                ("ip", C.c_int),
                ("vj0", C.c_int), ("vj1", C.c_int), ("vk0", C.c_int), ("vk1", C.c_int),
                ("lj0", C.c_int), ("lj1", C.c_int), ("lk0", C.c_int), ("lk1", C.c_int)]


class FdtdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_ERRNAMES.get(code, code)}: {msg}")
        self.code = code


# every symbol include/fdtd.h declares: name -> (restype, argtypes)
_dp = C.POINTER(C.c_double)
_vp = C.c_void_p
SYMBOLS = {
    "fdtd_create": (C.c_int, [C.c_int] * 3 + [C.c_double] * 4 + [C.c_int, C.POINTER(_vp)]),
    "fdtd_set_boundary": (C.c_int, [_vp, C.POINTER(C.c_int), _dp]),
    "fdtd_set_material_mode": (C.c_int, [_vp, C.c_int, C.c_int]),
    "fdtd_add_port": (C.c_int, [_vp, C.POINTER(fdtd_port), C.POINTER(C.c_int)]),
    "fdtd_set_dft": (C.c_int, [_vp, _dp, C.c_int]),
    "fdtd_set_option": (C.c_int, [_vp, C.c_int, C.c_long]),
    "fdtd_workspace_bytes": (C.c_size_t, [_vp]),
    "fdtd_commit": (C.c_int, [_vp, _vp, C.c_size_t, _vp]),
    "fdtd_set_materials_indexed": (C.c_int, [_vp, _vp, C.c_int, _dp, _dp, _dp]),
    "fdtd_set_materials_full": (C.c_int, [_vp, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_vp)]),
    "fdtd_step": (C.c_int, [_vp, C.c_long]),
    "fdtd_profile_step": (C.c_int, [_vp, C.c_long, _dp]),
    "fdtd_read_fields": (C.c_int, [_vp, C.c_int, _vp]),
    "fdtd_write_fields": (C.c_int, [_vp, C.c_int, _vp]),
    "fdtd_read_port_dft": (C.c_int, [_vp, C.c_int, _dp, _dp]),
    "fdtd_read_port_last": (C.c_int, [_vp, C.c_int, _dp, _dp]),
    "fdtd_reset": (C.c_int, [_vp]),
    "fdtd_step_count": (C.c_long, [_vp]),
    "fdtd_launch_count": (C.c_long, [_vp]),
    "fdtd_graph_replays": (C.c_long, [_vp]),
    "fdtd_device": (C.c_int, [_vp]),
    "fdtd_impl_name": (C.c_char_p, [_vp]),
    "fdtd_fused_kz": (C.c_int, [_vp]),
    "fdtd_two_step_box": (C.c_int, [_vp, C.POINTER(C.c_int)]),
    "fdtd_fused_tile": (C.c_int, [_vp]),
    "fdtd_set_z_interfaces": (C.c_int, [_vp, C.c_int, C.c_int]),
    "fdtd_step_begin": (C.c_int, [_vp]),
    "fdtd_step_end": (C.c_int, [_vp]),
    "fdtd_plane": (C.c_int, [_vp, C.c_int, C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)]),
    "fdtd_z_halo": (C.c_int, [_vp, C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
    "fdtd_z_link": (C.c_int, [_vp, C.c_int, C.POINTER(C.c_void_p), C.c_void_p]),
    "fdtd_last_error": (C.c_char_p, [_vp]),
    "fdtd_destroy": (None, [_vp]),
    "fdtd_port_probe_noalloc": (C.c_int, [_vp, _vp, _vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                          C.POINTER(fdtd_port), C.c_int, _vp, _vp, C.c_char_p, C.c_size_t]),
}
FDTD_NOALLOC_MAX_PORTS = 16

_lib = None


def lib():
    """Load (building first if the sources are newer) the CUDA library.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)  # AttributeError if the library does not export a declared symbol
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def library_path():
    return _build.LIB


def _check(h, code):
    if code != FDTD_OK:
        msg = lib().fdtd_last_error(h).decode() if h else ""
        raise FdtdError(code, msg)


def _ptr(a):
    """Address of a numpy array (host) or a torch tensor (host or CUDA); the object must be contiguous."""
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return a.data_ptr()
    raise TypeError("expected a numpy array or a torch tensor")


def _dbl(a):
    return None if a is None else np.ascontiguousarray(np.asarray(a, dtype=np.float64))


# ---- the C ABI, name for name ------------------------------------------------------------------------------------
def fdtd_create(nx, ny, nz, dx, dy, dz, dt, precision=FDTD_F32):
    h = _vp()
    code = lib().fdtd_create(int(nx), int(ny), int(nz), float(dx), float(dy), float(dz), float(dt), int(precision), C.byref(h))
    if code != FDTD_OK:
        raise FdtdError(code, "fdtd_create rejected the arguments (n < 2, d <= 0, bad precision, or dt above the CFL limit)")
    return h


def fdtd_set_boundary(h, pml_cells, cpml=None):
    p = (C.c_int * 6)(*[int(v) for v in pml_cells])
    c = _dbl(cpml)
    if c is not None and c.size != 6:
        raise ValueError("cpml must have 6 entries")
    _check(h, lib().fdtd_set_boundary(h, p, None if c is None else c.ctypes.data_as(_dp)))


def fdtd_set_material_mode(h, mode, has_mu=False):
    _check(h, lib().fdtd_set_material_mode(h, int(mode), int(bool(has_mu))))


def fdtd_add_port(h, port: dict) -> int:
    p = fdtd_port()
    for name, _ in fdtd_port._fields_:
        key = "is" if name == "is_" else name
        if key in port:
            setattr(p, name, port[key])
    pid = C.c_int(-1)
    _check(h, lib().fdtd_add_port(h, C.byref(p), C.byref(pid)))
    return pid.value


def fdtd_set_dft(h, freqs_hz):
    f = _dbl(freqs_hz).reshape(-1)
    _check(h, lib().fdtd_set_dft(h, f.ctypes.data_as(_dp), int(f.size)))


def fdtd_set_option(h, option, value):
    _check(h, lib().fdtd_set_option(h, int(option), int(value)))


def fdtd_workspace_bytes(h) -> int:
    return int(lib().fdtd_workspace_bytes(h))


def fdtd_commit(h, workspace, cuda_stream):
    """workspace: a CUDA uint8 tensor of >= fdtd_workspace_bytes(h) bytes; cuda_stream: integer cudaStream_t."""
    _check(h, lib().fdtd_commit(h, _ptr(workspace), int(workspace.numel() * workspace.element_size()), int(cuda_stream)))


def fdtd_set_materials_indexed(h, idx, eps_r, sigma, mu_r=None):
    e, s, m = _dbl(eps_r), _dbl(sigma), _dbl(mu_r)
    ne = e.size // 3
    if e.size != 3 * ne or s.size != e.size or (m is not None and m.size != e.size):
        raise ValueError("eps_r, sigma, mu_r must be [n_entries, 3]")
    if isinstance(idx, np.ndarray):
        idx = np.ascontiguousarray(idx, dtype=np.uint8)
    elif hasattr(idx, "element_size") and idx.element_size() != 1:
        raise ValueError("material index tensor must be uint8")
    _check(h, lib().fdtd_set_materials_indexed(h, _ptr(idx), ne, e.ctypes.data_as(_dp), s.ctypes.data_as(_dp),
                                                None if m is None else m.ctypes.data_as(_dp)))


def _check_cell_array(a, n_cells, itemsize, what):
    """A per-cell array handed over by address must hold n_cells elements of the handle's precision (the C side sees a
    bare pointer: a float64 array given to an fp32 handle would be reinterpreted silently)."""
    if isinstance(a, np.ndarray):
        size, isz, kind = a.size, a.dtype.itemsize, a.dtype.kind
    else:
        size, isz, kind = a.numel(), a.element_size(), ("f" if a.dtype.is_floating_point else "?")
    if kind != "f" or isz != itemsize or size != n_cells:
        raise ValueError(f"{what}: expected {n_cells} floating-point elements of {itemsize} bytes, got {size} x {isz} bytes ({kind})")


def fdtd_set_materials_full(h, eps_r, sigma, mu_r=None, n_cells=None, precision=None):
    """eps_r, sigma, mu_r: three arrays each (x, y, z component), host or device.  With n_cells and precision given (Solver
    passes them) every array is checked for element count, element type and contiguity before its address is used."""
    if n_cells is not None and precision is not None:
        for name, xs in (("eps_r", eps_r), ("sigma", sigma), ("mu_r", mu_r)):
            if xs is not None:
                if len(xs) != 3:
                    raise ValueError(f"{name}: three component arrays expected")
                for x in xs:
                    _check_cell_array(x, n_cells, 8 if precision == FDTD_F64 else 4, f"fdtd_set_materials_full {name}")

    def arr3(xs):
        return None if xs is None else (_vp * 3)(*[_ptr(x) for x in xs])
    _check(h, lib().fdtd_set_materials_full(h, arr3(eps_r), arr3(sigma), arr3(mu_r)))


def fdtd_step(h, n=1):
    _check(h, lib().fdtd_step(h, int(n)))


def fdtd_profile_step(h, n):
    """n steps with CUDA events between the kernels; returns ms per step of [H|fused, E, source, probes+DFT]."""
    ms = (C.c_double * 4)()
    _check(h, lib().fdtd_profile_step(h, int(n), ms))
    return list(ms)


def fdtd_read_fields(h, comp, dst):
    _check(h, lib().fdtd_read_fields(h, int(comp), _ptr(dst)))


def fdtd_write_fields(h, comp, src):
    _check(h, lib().fdtd_write_fields(h, int(comp), _ptr(src)))


def fdtd_read_port_dft(h, port, nf):
    V = np.zeros(2 * nf)
    I = np.zeros(2 * nf)
    _check(h, lib().fdtd_read_port_dft(h, int(port), V.ctypes.data_as(_dp), I.ctypes.data_as(_dp)))
    return V[0::2] + 1j * V[1::2], I[0::2] + 1j * I[1::2]


def fdtd_read_port_last(h, port):
    v, i = C.c_double(), C.c_double()
    _check(h, lib().fdtd_read_port_last(h, int(port), C.byref(v), C.byref(i)))
    return v.value, i.value


def fdtd_reset(h):
    _check(h, lib().fdtd_reset(h))


def fdtd_step_count(h) -> int:
    return int(lib().fdtd_step_count(h))


def fdtd_launch_count(h) -> int:
    return int(lib().fdtd_launch_count(h))


def fdtd_graph_replays(h) -> int:
    return int(lib().fdtd_graph_replays(h))


def fdtd_device(h) -> int:
    return int(lib().fdtd_device(h))


def fdtd_impl_name(h) -> str:
    return lib().fdtd_impl_name(h).decode()


def fdtd_fused_kz(h) -> int:
    return int(lib().fdtd_fused_kz(h))


def fdtd_fused_tile(h) -> int:
    return int(lib().fdtd_fused_tile(h))


def fdtd_two_step_box(h):
    box = (C.c_int * 6)()
    _check(h, lib().fdtd_two_step_box(h, box))
    return [int(v) for v in box]


def fdtd_set_z_interfaces(h, lo_open, hi_open):
    _check(h, lib().fdtd_set_z_interfaces(h, int(bool(lo_open)), int(bool(hi_open))))


def fdtd_step_begin(h):
    _check(h, lib().fdtd_step_begin(h))


def fdtd_step_end(h):
    _check(h, lib().fdtd_step_end(h))


def fdtd_plane(h, comp, k):
    """(device address, bytes) of the padded plane k in [-1, nz] of component comp in the current field set."""
    p, n = C.c_void_p(), C.c_size_t()
    _check(h, lib().fdtd_plane(h, int(comp), int(k), C.byref(p), C.byref(n)))
    return int(p.value), int(n.value)


def fdtd_z_halo(h, side):
    """([4 plane addresses: comp + 2 * set], counter address) a neighbour's kernels write for this slab's face `side`."""
    planes, flag = (C.c_void_p * 4)(), C.c_void_p()
    _check(h, lib().fdtd_z_halo(h, int(side), planes, C.byref(flag)))
    return [int(p) for p in planes], int(flag.value)


def fdtd_z_link(h, side, peer_planes, peer_flag):
    """Give this slab the fdtd_z_halo answer (addresses valid in THIS process) of its neighbour on `side`."""
    _check(h, lib().fdtd_z_link(h, int(side), (C.c_void_p * 4)(*[int(p) for p in peer_planes]), C.c_void_p(int(peer_flag))))


def fdtd_last_error(h) -> str:
    return lib().fdtd_last_error(h).decode()


def fdtd_destroy(h):
    lib().fdtd_destroy(h)


def fdtd_port_probe_noalloc(Ez, Hy, Hz, precision, nx, ny, nz, dy, dz, ports, VI, cuda_stream):
    """V and I (Eq. 4) of `ports` from three CUDA field tensors of nx*ny*nz elements, written into the CUDA float64 tensor
    VI (2 per port: V, I) on the given stream.  This is the entry point for callers that cannot allocate device memory (a
    monitor beside a running solver, a plug-in in a host that owns all GPU memory, a no-allocation region): the hand-over
    memory of the reduction is a fixed array inside the library, shared by every call on a GPU -- so at most
    FDTD_NOALLOC_MAX_PORTS ports per call, and calls that overlap on one GPU race.  Nothing is allocated here either: the
    tensors are the caller's, the port list is marshalled into host memory."""
    n_cells = int(nx) * int(ny) * int(nz)
    for name, t in (("Ez", Ez), ("Hy", Hy), ("Hz", Hz)):
        _check_cell_array(t, n_cells, 8 if precision == FDTD_F64 else 4, f"fdtd_port_probe_noalloc {name}")
    _check_cell_array(VI, 2 * len(ports), 8, "fdtd_port_probe_noalloc VI")
    arr = (fdtd_port * max(len(ports), 1))()
    for q, port in zip(arr, ports):
        for name, _ in fdtd_port._fields_:
            key = "is" if name == "is_" else name
            if key in port:
                setattr(q, name, port[key])
    err = C.create_string_buffer(256)
    code = lib().fdtd_port_probe_noalloc(_ptr(Ez), _ptr(Hy), _ptr(Hz), int(precision), int(nx), int(ny), int(nz), float(dy),
                                         float(dz), arr, len(ports), _ptr(VI), int(cuda_stream), err, len(err))
    if code != FDTD_OK:
        raise FdtdError(code, err.value.decode())
