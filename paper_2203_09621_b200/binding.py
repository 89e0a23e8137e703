"""ctypes binding of include/dmpt.h: same names, argument marshalling only.

`lib()` loads the in-tree `libdmpt.so` and fails loudly when it is missing (build it with
`python -m paper_2203_09621_b200.build` or `__graft_entry__.build()`); nothing here computes.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, field

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdmpt.so")

EXPORTED_SYMBOLS = (
    "dmpt_default_options", "dmpt_workspace_bytes", "dmpt_create", "dmpt_set_hamiltonian",
    "dmpt_run", "dmpt_run_host", "dmpt_layer_products", "dmpt_destroy", "dmpt_strerror",
    "dmpt_last_cuda_error", "dmpt_spectral_bounds", "dmpt_initial_transform", "dmpt_split",
    "dmpt_layer_products2", "dmpt_product_nt", "dmpt_inverse_factor", "dmpt_workspace_bytes_fields", "dmpt_set_hamiltonian_fields", "dmpt_run_fields",
    "dmpt_run_orders", "dmpt_layer_products3", "dmpt_congruence", "dmpt_fd_response",
    "dmpt_run_fields_host",
    "dmpt_pair_workspace_bytes", "dmpt_pair_create", "dmpt_pair_set_hamiltonian", "dmpt_pair_run", "dmpt_pair_destroy",
    "dmpt_pair_last_cuda_error",
    "dmpt_spectral_bounds_noalloc",
)

DMPT_OK, DMPT_EINVAL, DMPT_ESTATE, DMPT_ECUDA = 0, -1, -2, -3
DMPT_EDEGENERATE, DMPT_ENOCONV, DMPT_ENUMERIC, DMPT_EWORKSPACE = -4, -5, -6, -7
DMPT_ELIMIT = -8
DMPT_NOALLOC_MAX_N = 65536


class DmptOptions(C.Structure):
    _fields_ = [
        ("max_layers", C.c_int), ("order", C.c_int), ("s0_shift", C.c_int),
        ("s1_autoscale", C.c_int), ("bounds", C.c_int),
        ("eps_min", C.c_double), ("eps_max", C.c_double),
        ("wave_sync", C.c_int), ("num_fields", C.c_int), ("epilogue_direct", C.c_int), ("lanczos_steps", C.c_int),
        ("no_pdl", C.c_int), ("loop_graph", C.c_int),
        ("order0_narrow", C.c_int), ("reserved", C.c_int * 1),
    ]


class _CResult(C.Structure):
    _fields_ = [
        ("status", C.c_int), ("layers", C.c_int), ("layers_d0", C.c_int), ("layers_d1", C.c_int),
        ("launches", C.c_int), ("layers_d2", C.c_int), ("layers_d3", C.c_int), ("reserved_i", C.c_int * 1),
        ("eps_min", C.c_double), ("eps_max", C.c_double), ("fro_err0", C.c_double),
        ("ms_total", C.c_double), ("ms_loop", C.c_double), ("ms_bounds", C.c_double),
        ("ms_transform", C.c_double), ("ms_split", C.c_double), ("sm_clock_mhz", C.c_double),
        ("sigma", C.POINTER(C.c_int8)), ("tr_s", C.POINTER(C.c_double)), ("tr_x", C.POINTER(C.c_double)),
        ("id_err", C.POINTER(C.c_double)), ("fro_err1", C.POINTER(C.c_double)),
        ("fro_err2", C.POINTER(C.c_double)), ("fro_err3", C.POINTER(C.c_double)),
    ]


class DmptError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        msg = f"{where}: {dmpt_strerror(code)} ({code})"
        if detail:
            msg += f" - {detail}"
        super().__init__(msg)


_lib = None


def lib():
    """The loaded C-ABI library.  Raises if it has not been built: there is no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build the CUDA extension first "
                "(python -m paper_2203_09621_b200.build). There is no CPU fallback.")
        L = C.CDLL(LIB_PATH)
        L.dmpt_default_options.argtypes = [C.POINTER(DmptOptions)]
        L.dmpt_default_options.restype = None
        L.dmpt_workspace_bytes.argtypes = [C.c_int, C.c_int]
        L.dmpt_workspace_bytes.restype = C.c_size_t
        L.dmpt_workspace_bytes_fields.argtypes = [C.c_int, C.c_int]
        L.dmpt_workspace_bytes_fields.restype = C.c_size_t
        L.dmpt_set_hamiltonian_fields.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p), C.c_int, C.c_int]
        L.dmpt_set_hamiltonian_fields.restype = C.c_int
        L.dmpt_run_fields.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p), C.c_int, C.POINTER(_CResult)]
        L.dmpt_run_fields.restype = C.c_int
        L.dmpt_run_orders.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.c_int, C.POINTER(_CResult)]
        L.dmpt_run_orders.restype = C.c_int
        L.dmpt_layer_products3.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int,
                                           C.c_void_p, C.c_int]
        L.dmpt_layer_products3.restype = C.c_int
        L.dmpt_run_fields_host.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_void_p,
                                           C.POINTER(C.c_void_p), C.c_int, C.POINTER(_CResult)]
        L.dmpt_run_fields_host.restype = C.c_int
        L.dmpt_congruence.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int]
        L.dmpt_congruence.restype = C.c_int
        L.dmpt_spectral_bounds_noalloc.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.dmpt_spectral_bounds_noalloc.restype = C.c_int
        L.dmpt_fd_response.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_int,
                                       C.c_void_p, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_double)]
        L.dmpt_fd_response.restype = C.c_int
        L.dmpt_pair_workspace_bytes.argtypes = [C.c_int, C.c_int]
        L.dmpt_pair_workspace_bytes.restype = C.c_size_t
        L.dmpt_pair_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.POINTER(DmptOptions), C.c_int, C.c_void_p,
                                       C.c_size_t, C.c_int, C.c_void_p, C.c_size_t]
        L.dmpt_pair_create.restype = C.c_int
        L.dmpt_pair_set_hamiltonian.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        L.dmpt_pair_set_hamiltonian.restype = C.c_int
        L.dmpt_pair_run.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.POINTER(_CResult)]
        L.dmpt_pair_run.restype = C.c_int
        L.dmpt_pair_destroy.argtypes = [C.c_void_p]
        L.dmpt_pair_destroy.restype = C.c_int
        L.dmpt_pair_last_cuda_error.argtypes = [C.c_void_p]
        L.dmpt_pair_last_cuda_error.restype = C.c_char_p
        L.dmpt_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.POINTER(DmptOptions), C.c_void_p,
                                  C.c_size_t, C.c_void_p]
        L.dmpt_create.restype = C.c_int
        L.dmpt_set_hamiltonian.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        L.dmpt_set_hamiltonian.restype = C.c_int
        L.dmpt_run.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.POINTER(_CResult)]
        L.dmpt_run.restype = C.c_int
        L.dmpt_run_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p,
                                    C.c_void_p, C.c_void_p, C.c_int, C.POINTER(_CResult)]
        L.dmpt_run_host.restype = C.c_int
        L.dmpt_layer_products.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                          C.c_void_p, C.c_int]
        L.dmpt_layer_products.restype = C.c_int
        L.dmpt_layer_products2.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                           C.c_int]
        L.dmpt_layer_products2.restype = C.c_int
        L.dmpt_product_nt.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int]
        L.dmpt_product_nt.restype = C.c_int
        L.dmpt_inverse_factor.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_double,
                                          C.POINTER(C.c_int), C.POINTER(C.c_double)]
        L.dmpt_inverse_factor.restype = C.c_int
        L.dmpt_spectral_bounds.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_double),
                                           C.POINTER(C.c_double)]
        L.dmpt_spectral_bounds.restype = C.c_int
        L.dmpt_initial_transform.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double,
                                             C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_double)]
        L.dmpt_initial_transform.restype = C.c_int
        L.dmpt_split.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int]
        L.dmpt_split.restype = C.c_int
        L.dmpt_destroy.argtypes = [C.c_void_p]
        L.dmpt_destroy.restype = C.c_int
        L.dmpt_strerror.argtypes = [C.c_int]
        L.dmpt_strerror.restype = C.c_char_p
        L.dmpt_last_cuda_error.argtypes = [C.c_void_p]
        L.dmpt_last_cuda_error.restype = C.c_char_p
        _lib = L
    return _lib


# ------------------------------------------------------------------ same-name thin wrappers
def dmpt_default_options() -> DmptOptions:
    o = DmptOptions()
    lib().dmpt_default_options(C.byref(o))
    return o


def dmpt_workspace_bytes(n: int, order: int = 1) -> int:
    return int(lib().dmpt_workspace_bytes(int(n), int(order)))


def dmpt_workspace_bytes_fields(n: int, num_fields: int) -> int:
    return int(lib().dmpt_workspace_bytes_fields(int(n), int(num_fields)))


def dmpt_set_hamiltonian_fields(ctx, h0_ptr: int, h1_ptrs, ld: int, n_occ: int) -> None:
    arr = (C.c_void_p * len(h1_ptrs))(*[C.c_void_p(p) for p in h1_ptrs])
    rc = lib().dmpt_set_hamiltonian_fields(ctx, C.c_void_p(h0_ptr), arr, int(ld), int(n_occ))
    if rc != DMPT_OK:
        raise DmptError(rc, "dmpt_set_hamiltonian_fields")


def dmpt_run_fields(ctx, d0_ptr: int, d1_ptrs, ld: int, res) -> int:
    arr = (C.c_void_p * len(d1_ptrs))(*[C.c_void_p(p) for p in d1_ptrs])
    return int(lib().dmpt_run_fields(ctx, C.c_void_p(d0_ptr), arr, int(ld), C.byref(res) if res is not None else None))


def dmpt_run_orders(ctx, d_ptrs, ld: int, res) -> int:
    arr = (C.c_void_p * len(d_ptrs))(*[C.c_void_p(p) for p in d_ptrs])
    return int(lib().dmpt_run_orders(ctx, arr, int(ld), C.byref(res) if res is not None else None))


def dmpt_layer_products3(ctx, s0_ptr, s1_ptr, s2_ptr, s3_ptr, ld, x3_ptr, ld_out) -> int:
    return int(lib().dmpt_layer_products3(ctx, C.c_void_p(s0_ptr), C.c_void_p(s1_ptr), C.c_void_p(s2_ptr),
                                          C.c_void_p(s3_ptr), int(ld), C.c_void_p(x3_ptr), int(ld_out)))


def dmpt_run_fields_host(ctx, h0_ptr, h1_ptrs, ld_in, n_occ, d0_ptr, d1_ptrs, ld_out, res) -> int:
    a = (C.c_void_p * len(h1_ptrs))(*[C.c_void_p(p) for p in h1_ptrs])
    b = (C.c_void_p * len(d1_ptrs))(*[C.c_void_p(p) for p in d1_ptrs])
    return int(lib().dmpt_run_fields_host(ctx, C.c_void_p(h0_ptr), a, int(ld_in), int(n_occ), C.c_void_p(d0_ptr), b,
                                          int(ld_out), C.byref(res) if res is not None else None))


def dmpt_congruence(ctx, z_ptr, x_ptr, ld, transpose_z, c_ptr, ld_out) -> int:
    return int(lib().dmpt_congruence(ctx, C.c_void_p(z_ptr), C.c_void_p(x_ptr), int(ld), int(transpose_z),
                                     C.c_void_p(c_ptr), int(ld_out)))


def dmpt_fd_response(ctx, h0_ptr, h1_ptr, ld, n_occ, h, points, d1_ptr, ld_out):
    layers = (C.c_int * 4)()
    ms = C.c_double()
    rc = int(lib().dmpt_fd_response(ctx, C.c_void_p(h0_ptr), C.c_void_p(h1_ptr), int(ld), int(n_occ), float(h),
                                    int(points), C.c_void_p(d1_ptr), int(ld_out), layers, C.byref(ms)))
    return rc, list(layers[:int(points)]) if points in (2, 4) else [], ms.value


def dmpt_pair_workspace_bytes(n: int, side: int) -> int:
    return int(lib().dmpt_pair_workspace_bytes(int(n), int(side)))


def dmpt_pair_create(n, opt, device0, ws0_ptr, ws0_bytes, device1, ws1_ptr, ws1_bytes):
    h = C.c_void_p()
    rc = lib().dmpt_pair_create(C.byref(h), int(n), C.byref(opt) if opt is not None else None, int(device0),
                                C.c_void_p(ws0_ptr), int(ws0_bytes), int(device1), C.c_void_p(ws1_ptr), int(ws1_bytes))
    if rc != DMPT_OK:
        raise DmptError(rc, "dmpt_pair_create")
    return h


def dmpt_pair_set_hamiltonian(pair, h0_ptr, h1_ptr, ld, n_occ) -> None:
    rc = lib().dmpt_pair_set_hamiltonian(pair, C.c_void_p(h0_ptr), C.c_void_p(h1_ptr), int(ld), int(n_occ))
    if rc != DMPT_OK:
        raise DmptError(rc, "dmpt_pair_set_hamiltonian")


def dmpt_pair_run(pair, d0_ptr, d1_ptr, ld, res) -> int:
    return int(lib().dmpt_pair_run(pair, C.c_void_p(d0_ptr), C.c_void_p(d1_ptr), int(ld),
                                   C.byref(res) if res is not None else None))


def dmpt_pair_destroy(pair) -> None:
    lib().dmpt_pair_destroy(pair)


def dmpt_pair_last_cuda_error(pair) -> str:
    return lib().dmpt_pair_last_cuda_error(pair).decode()


def dmpt_strerror(code: int) -> str:
    return lib().dmpt_strerror(int(code)).decode()


def dmpt_last_cuda_error(ctx) -> str:
    return lib().dmpt_last_cuda_error(ctx).decode()


def dmpt_create(n: int, opt: DmptOptions | None, workspace_ptr: int, workspace_bytes: int, stream_ptr: int = 0):
    h = C.c_void_p()
    rc = lib().dmpt_create(C.byref(h), int(n), C.byref(opt) if opt is not None else None,
                           C.c_void_p(workspace_ptr), int(workspace_bytes), C.c_void_p(stream_ptr))
    if rc != DMPT_OK:
        raise DmptError(rc, "dmpt_create")
    return h


def dmpt_set_hamiltonian(ctx, h0_ptr: int, h1_ptr: int, ld: int, n_occ: int) -> None:
    rc = lib().dmpt_set_hamiltonian(ctx, C.c_void_p(h0_ptr), C.c_void_p(h1_ptr), int(ld), int(n_occ))
    if rc != DMPT_OK:
        raise DmptError(rc, "dmpt_set_hamiltonian")


def dmpt_run(ctx, d0_ptr: int, d1_ptr: int, d2_ptr: int, ld: int, res: _CResult | None) -> int:
    return int(lib().dmpt_run(ctx, C.c_void_p(d0_ptr), C.c_void_p(d1_ptr), C.c_void_p(d2_ptr or None),
                              int(ld), C.byref(res) if res is not None else None))


def dmpt_run_host(ctx, h0_ptr, h1_ptr, ld_in, n_occ, d0_ptr, d1_ptr, d2_ptr, ld_out, res) -> int:
    return int(lib().dmpt_run_host(ctx, C.c_void_p(h0_ptr), C.c_void_p(h1_ptr), int(ld_in), int(n_occ),
                                   C.c_void_p(d0_ptr), C.c_void_p(d1_ptr), C.c_void_p(d2_ptr or None),
                                   int(ld_out), C.byref(res) if res is not None else None))


def dmpt_layer_products(ctx, s0_ptr, s1_ptr, ld, x0_ptr, x1_ptr, ld_out) -> int:
    return int(lib().dmpt_layer_products(ctx, C.c_void_p(s0_ptr), C.c_void_p(s1_ptr), int(ld),
                                         C.c_void_p(x0_ptr), C.c_void_p(x1_ptr), int(ld_out)))


def dmpt_layer_products2(ctx, s0_ptr, s1_ptr, s2_ptr, ld, x2_ptr, ld_out) -> int:
    return int(lib().dmpt_layer_products2(ctx, C.c_void_p(s0_ptr), C.c_void_p(s1_ptr), C.c_void_p(s2_ptr), int(ld),
                                          C.c_void_p(x2_ptr), int(ld_out)))


def dmpt_product_nt(ctx, a_ptr, b_ptr, ld, c_ptr, ld_out) -> int:
    return int(lib().dmpt_product_nt(ctx, C.c_void_p(a_ptr), C.c_void_p(b_ptr), int(ld), C.c_void_p(c_ptr), int(ld_out)))


def dmpt_inverse_factor(ctx, s_ptr, ld, z_ptr, ld_z, max_iter, tol):
    it, err = C.c_int(), C.c_double()
    rc = int(lib().dmpt_inverse_factor(ctx, C.c_void_p(s_ptr), int(ld), C.c_void_p(z_ptr), int(ld_z), int(max_iter),
                                       float(tol), C.byref(it), C.byref(err)))
    return rc, it.value, err.value


def dmpt_spectral_bounds(ctx, h0_ptr, ld):
    lo, hi = C.c_double(), C.c_double()
    rc = int(lib().dmpt_spectral_bounds(ctx, C.c_void_p(h0_ptr), int(ld), C.byref(lo), C.byref(hi)))
    return rc, lo.value, hi.value


def dmpt_spectral_bounds_noalloc(h0_ptr, n, ld, eps_ptr, stream=0) -> int:
    """Context-free a1 with static scratch (include/dmpt.h): device pointers in, two device doubles out, stream-ordered."""
    return int(lib().dmpt_spectral_bounds_noalloc(C.c_void_p(h0_ptr), int(n), int(ld), C.c_void_p(eps_ptr),
                                                  C.c_void_p(stream)))


def spectral_bounds_noalloc(h0, out, stream=None):
    """Gershgorin bounds of the CUDA fp32 matrix `h0` into `out` (CUDA float64, two elements: eps_min, eps_max), enqueued
    on `stream` (torch stream; default: the current one) with no allocation on either side.  `out` is returned; it is
    valid once the stream has reached this point.  n > DMPT_NOALLOC_MAX_N raises DmptError(DMPT_ELIMIT)."""
    import torch

    if h0.dim() != 2 or h0.shape[0] != h0.shape[1] or h0.dtype != torch.float32 or h0.stride(1) != 1 or not h0.is_cuda:
        raise ValueError("h0: a square CUDA fp32 matrix with unit column stride is required")
    if out.dtype != torch.float64 or out.numel() < 2 or not out.is_contiguous() or out.device != h0.device:
        raise ValueError("out: two contiguous float64 elements on h0's device are required")
    with torch.cuda.device(h0.device):
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = dmpt_spectral_bounds_noalloc(h0.data_ptr(), h0.shape[0], h0.stride(0) if h0.shape[0] > 1 else 1,
                                          out.data_ptr(), st.cuda_stream)
    if rc != DMPT_OK:
        raise DmptError(rc, "dmpt_spectral_bounds_noalloc")
    return out


def dmpt_initial_transform(ctx, h0_ptr, h1_ptr, ld, eps_min, eps_max, s0_ptr, s1_ptr, ld_out):
    tr = C.c_double()
    rc = int(lib().dmpt_initial_transform(ctx, C.c_void_p(h0_ptr), C.c_void_p(h1_ptr), int(ld), float(eps_min),
                                          float(eps_max), C.c_void_p(s0_ptr), C.c_void_p(s1_ptr), int(ld_out),
                                          C.byref(tr)))
    return rc, tr.value


def dmpt_split(ctx, x_ptr, ld, shift, diag_half, hi_ptr, lo_ptr, ld_out) -> int:
    return int(lib().dmpt_split(ctx, C.c_void_p(x_ptr), int(ld), int(shift), int(diag_half), C.c_void_p(hi_ptr),
                                C.c_void_p(lo_ptr), int(ld_out)))


def dmpt_destroy(ctx) -> None:
    lib().dmpt_destroy(ctx)


# ------------------------------------------------------------------ convenience object
@dataclass
class DmptResult:
    status: int
    layers: int
    layers_d0: int
    layers_d1: int
    launches: int
    eps_min: float
    eps_max: float
    fro_err0: float
    ms_total: float
    ms_loop: float
    ms_bounds: float = 0.0
    ms_transform: float = 0.0
    ms_split: float = 0.0
    sm_clock_mhz: float = 0.0     # SM clock of the layer loop from the device's own counters (include/dmpt.h)
    layers_d2: int = 0
    sigma: list = field(default_factory=list)
    tr_s: list = field(default_factory=list)
    tr_x: list = field(default_factory=list)
    id_err: list = field(default_factory=list)
    fro_err1: list = field(default_factory=list)
    fro_err2: list = field(default_factory=list)
    fro_err3: list = field(default_factory=list)
    layers_d3: int = 0
    d0: object = None
    d1: object = None
    d2: object = None
    d3: object = None


class Dmpt:
    """Owns a dmpt_ctx plus the torch-allocated workspace.  Marshalling only."""

    def __init__(self, n, order=1, max_layers=200, s0_shift=-1, s1_autoscale=True, bounds=None,
                 device="cuda:0", stream=None, wave_sync=True, num_fields=1, epilogue_direct=False, lanczos_steps=0,
                 pdl=True, loop_graph=False, order0_narrow=False):
        import torch

        self.torch = torch
        self.n = int(n)
        self.order = int(order)
        self.device = torch.device(device)
        if self.device.type != "cuda":
            raise DmptError(DMPT_ECUDA, "Dmpt", "a CUDA device is required; there is no CPU path")
        opt = dmpt_default_options()
        opt.max_layers = int(max_layers)
        opt.order = self.order
        opt.s0_shift = int(s0_shift)
        opt.s1_autoscale = 1 if s1_autoscale else 0
        opt.wave_sync = 1 if wave_sync else 0
        opt.num_fields = int(num_fields)
        opt.epilogue_direct = 1 if epilogue_direct else 0
        opt.no_pdl = 0 if pdl else 1
        opt.loop_graph = 1 if loop_graph else 0
        opt.order0_narrow = 1 if order0_narrow else 0
        self.num_fields = int(num_fields)
        if isinstance(bounds, str):
            if bounds != "lanczos":
                raise DmptError(DMPT_EINVAL, "Dmpt", "bounds: None (Gershgorin), (eps_min, eps_max) or 'lanczos'")
            opt.bounds = 2
            opt.lanczos_steps = int(lanczos_steps)
        elif bounds is not None:
            opt.bounds = 1
            opt.eps_min, opt.eps_max = float(bounds[0]), float(bounds[1])
        # size the per-layer record buffers as the library does (dmpt_create: <= 0 -> 200, capped at 1024)
        if opt.max_layers <= 0:
            opt.max_layers = 200
        opt.max_layers = min(opt.max_layers, 1024)
        self.max_layers = opt.max_layers
        nbytes = (dmpt_workspace_bytes_fields(self.n, self.num_fields) if self.num_fields > 1
                  else dmpt_workspace_bytes(self.n, self.order))
        if nbytes == 0:
            raise DmptError(DMPT_EINVAL, "dmpt_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.ctx = dmpt_create(self.n, opt, self.workspace.data_ptr(), nbytes, self.stream.cuda_stream)
        self._h = None

    def set_hamiltonian(self, h0, h1, n_occ):
        t = self.torch
        for m in (h0, h1):
            if m is None and self.order == 0:
                continue                # ground-state mode takes no perturbation
            if m is None or not (m.is_cuda and m.dtype == t.float32 and m.dim() == 2 and m.stride(1) == 1):
                raise DmptError(DMPT_EINVAL, "set_hamiltonian", "need row-major fp32 CUDA matrices")
        if h1 is not None and h1.stride(0) != h0.stride(0):
            raise DmptError(DMPT_EINVAL, "set_hamiltonian", "h0 and h1 need the same leading dimension")
        self._h = (h0, h1)          # keep the storage alive
        dmpt_set_hamiltonian(self.ctx, h0.data_ptr(), h1.data_ptr() if h1 is not None else 0, h0.stride(0), n_occ)

    def _new_result(self):
        ml = self.max_layers
        bufs = dict(sigma=(C.c_int8 * ml)(), tr_s=(C.c_double * ml)(), tr_x=(C.c_double * ml)(),
                    id_err=(C.c_double * ml)(), fro_err1=(C.c_double * ml)(), fro_err2=(C.c_double * ml)(),
                    fro_err3=(C.c_double * ml)())
        r = _CResult()
        r.sigma = C.cast(bufs["sigma"], C.POINTER(C.c_int8))
        for k in ("tr_s", "tr_x", "id_err", "fro_err1", "fro_err2", "fro_err3"):
            setattr(r, k, C.cast(bufs[k], C.POINTER(C.c_double)))
        return r, bufs

    def _wrap(self, rc, r, bufs, d0, d1, d2, check):
        if rc not in (DMPT_OK, DMPT_ENOCONV) and check:
            raise DmptError(rc, "dmpt_run", dmpt_last_cuda_error(self.ctx))
        nl = max(0, int(r.layers))
        return DmptResult(status=rc, layers=r.layers, layers_d0=r.layers_d0, layers_d1=r.layers_d1,
                          launches=r.launches, eps_min=r.eps_min, eps_max=r.eps_max, fro_err0=r.fro_err0,
                          ms_total=r.ms_total, ms_loop=r.ms_loop, ms_bounds=r.ms_bounds,
                          ms_transform=r.ms_transform, ms_split=r.ms_split, sm_clock_mhz=r.sm_clock_mhz,
                          sigma=list(bufs["sigma"][:nl]), tr_s=list(bufs["tr_s"][:nl]),
                          tr_x=list(bufs["tr_x"][:nl]), id_err=list(bufs["id_err"][:nl]),
                          fro_err1=list(bufs["fro_err1"][:nl]),
                          fro_err2=list(bufs["fro_err2"][:nl]) if (self.order >= 2 or self.num_fields > 1) else [],
                          fro_err3=list(bufs["fro_err3"][:nl]) if (self.num_fields > 2 or self.order == 3) else [],
                          layers_d2=r.layers_d2, layers_d3=r.layers_d3, d0=d0, d1=d1, d2=d2)

    def _check_outputs(self, where, cuda, *mats):
        """The C ABI takes ONE leading dimension for all outputs: refuse views that disagree."""
        t = self.torch
        ms = [m for m in mats if m is not None]
        for m in ms:
            if not (m.is_cuda == cuda and m.dtype == t.float32 and m.dim() == 2 and m.stride(1) == 1
                    and m.stride(0) == ms[0].stride(0) and m.shape[0] >= self.n and m.shape[1] >= self.n):
                raise DmptError(DMPT_EINVAL, where, "outputs must be row-major fp32 matrices with one leading dimension")

    def run(self, out=None, check=True) -> DmptResult:
        t = self.torch
        n = self.n
        if out is None:
            d0 = t.empty((n, n), dtype=t.float32, device=self.device)
            d1 = t.empty((n, n), dtype=t.float32, device=self.device) if self.order >= 1 else None
        else:
            d0, d1 = out[0], (out[1] if len(out) > 1 else None)
        if self.order != 2:
            d2 = None
        elif out is not None and len(out) > 2:
            d2 = out[2]
        else:
            d2 = t.empty((n, n), dtype=t.float32, device=self.device)
        self._check_outputs("run", True, d0, d1, d2)
        r, bufs = self._new_result()
        rc = dmpt_run(self.ctx, d0.data_ptr(), d1.data_ptr() if d1 is not None else 0,
                      d2.data_ptr() if d2 is not None else 0, d0.stride(0), r)
        return self._wrap(rc, r, bufs, d0, d1, d2, check)

    def run_orders(self, check=True) -> DmptResult:
        """D0 .. D_order through dmpt_run_orders (any supported order; the only run call for order 3)."""
        t = self.torch
        n = self.n
        ds = [t.empty((n, n), dtype=t.float32, device=self.device) for _ in range(self.order + 1)]
        r, bufs = self._new_result()
        rc = dmpt_run_orders(self.ctx, [m.data_ptr() for m in ds], n, r)
        ds += [None] * (4 - len(ds))
        out = self._wrap(rc, r, bufs, ds[0], ds[1], ds[2], check)
        out.d3 = ds[3]
        return out

    def layer_products3(self, s0, s1, s2, s3):
        t = self.torch
        x3 = t.empty((self.n, self.n), dtype=t.float32, device=self.device)
        rc = dmpt_layer_products3(self.ctx, s0.data_ptr(), s1.data_ptr(), s2.data_ptr(), s3.data_ptr(), s0.stride(0),
                                  x3.data_ptr(), self.n)
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_layer_products3", dmpt_last_cuda_error(self.ctx))
        return x3

    def set_hamiltonian_fields(self, h0, h1s, n_occ):
        """h1s: num_fields perturbations sharing h0 (row-major fp32 CUDA matrices with h0's leading dimension)."""
        t = self.torch
        h1s = list(h1s)
        for m in [h0] + h1s:
            if not (m.is_cuda and m.dtype == t.float32 and m.dim() == 2 and m.stride(1) == 1
                    and m.stride(0) == h0.stride(0)):
                raise DmptError(DMPT_EINVAL, "set_hamiltonian_fields", "need row-major fp32 CUDA matrices, one ld")
        if len(h1s) != self.num_fields:
            raise DmptError(DMPT_EINVAL, "set_hamiltonian_fields", f"need {self.num_fields} perturbations")
        self._h = (h0, h1s)
        dmpt_set_hamiltonian_fields(self.ctx, h0.data_ptr(), [m.data_ptr() for m in h1s], h0.stride(0), n_occ)

    def run_fields(self, check=True) -> DmptResult:
        """D0 and one D1 per field; the result's d1 is the list of them."""
        t = self.torch
        n = self.n
        d0 = t.empty((n, n), dtype=t.float32, device=self.device)
        d1s = [t.empty((n, n), dtype=t.float32, device=self.device) for _ in range(self.num_fields)]
        r, bufs = self._new_result()
        rc = dmpt_run_fields(self.ctx, d0.data_ptr(), [m.data_ptr() for m in d1s], n, r)
        return self._wrap(rc, r, bufs, d0, d1s, None, check)

    def run_fields_host(self, h0, h1s, n_occ, out=None, check=True) -> DmptResult:
        """h0, h1s: CPU fp32 tensors (pinned recommended) with one leading dimension; out = (d0, [d1_f]) CPU tensors."""
        t = self.torch
        n = self.n
        h1s = list(h1s)
        if len(h1s) != self.num_fields or any(m.stride(0) != h0.stride(0) for m in h1s):
            raise DmptError(DMPT_EINVAL, "run_fields_host", f"need {self.num_fields} perturbations with h0's leading dimension")
        if out is None:
            d0 = t.empty((n, n), dtype=t.float32, pin_memory=True)
            d1s = [t.empty((n, n), dtype=t.float32, pin_memory=True) for _ in range(self.num_fields)]
        else:
            d0, d1s = out[0], list(out[1])
        self._check_outputs("run_fields_host", False, d0, *d1s)
        r, bufs = self._new_result()
        rc = dmpt_run_fields_host(self.ctx, h0.data_ptr(), [m.data_ptr() for m in h1s], h0.stride(0), n_occ,
                                  d0.data_ptr(), [m.data_ptr() for m in d1s], d0.stride(0), r)
        return self._wrap(rc, r, bufs, d0, d1s, None, check)

    def run_host(self, h0, h1, n_occ, out=None, check=True) -> DmptResult:
        """h0, h1: CPU fp32 tensors (pinned recommended); outputs are CPU tensors."""
        t = self.torch
        n = self.n
        if out is None:
            d0 = t.empty((n, n), dtype=t.float32, pin_memory=True)
            d1 = t.empty((n, n), dtype=t.float32, pin_memory=True) if self.order >= 1 else None
        else:
            d0, d1 = out[0], (out[1] if len(out) > 1 else None)
        if self.order != 2:
            d2 = None
        elif out is not None and len(out) > 2:
            d2 = out[2]
        else:
            d2 = t.empty((n, n), dtype=t.float32, pin_memory=True)
        if h1 is not None and h1.stride(0) != h0.stride(0):
            raise DmptError(DMPT_EINVAL, "run_host", "h0 and h1 need the same leading dimension")
        self._check_outputs("run_host", False, d0, d1, d2)
        r, bufs = self._new_result()
        rc = dmpt_run_host(self.ctx, h0.data_ptr(), h1.data_ptr() if h1 is not None else 0, h0.stride(0), n_occ,
                           d0.data_ptr(), d1.data_ptr() if d1 is not None else 0,
                           d2.data_ptr() if d2 is not None else 0, d0.stride(0), r)
        return self._wrap(rc, r, bufs, d0, d1, d2, check)

    def layer_products(self, s0, s1):
        t = self.torch
        n = self.n
        x0 = t.empty((n, n), dtype=t.float32, device=self.device)
        x1 = t.empty((n, n), dtype=t.float32, device=self.device)
        rc = dmpt_layer_products(self.ctx, s0.data_ptr(), s1.data_ptr(), s0.stride(0), x0.data_ptr(),
                                 x1.data_ptr(), n)
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_layer_products", dmpt_last_cuda_error(self.ctx))
        return x0, x1

    def layer_products2(self, s0, s1, s2):
        t = self.torch
        x2 = t.empty((self.n, self.n), dtype=t.float32, device=self.device)
        rc = dmpt_layer_products2(self.ctx, s0.data_ptr(), s1.data_ptr(), s2.data_ptr(), s0.stride(0),
                                  x2.data_ptr(), self.n)
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_layer_products2", dmpt_last_cuda_error(self.ctx))
        return x2

    def product_nt(self, a, b):
        """C = a @ b.T in the dual half-precision representation (general matrices)."""
        t = self.torch
        c = t.empty((self.n, self.n), dtype=t.float32, device=self.device)
        if a.stride(0) != b.stride(0):
            raise DmptError(DMPT_EINVAL, "product_nt", "a and b need the same leading dimension")
        rc = dmpt_product_nt(self.ctx, a.data_ptr(), b.data_ptr(), a.stride(0), c.data_ptr(), self.n)
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_product_nt", dmpt_last_cuda_error(self.ctx))
        return c

    def inverse_factor(self, s, max_iter=30, tol=0.0):
        """(Z, iterations, ||Z^T S Z - I||_F) for a symmetric positive definite overlap matrix s."""
        t = self.torch
        z = t.empty((self.n, self.n), dtype=t.float32, device=self.device)
        rc, it, err = dmpt_inverse_factor(self.ctx, s.data_ptr(), s.stride(0), z.data_ptr(), self.n, max_iter, tol)
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_inverse_factor", dmpt_last_cuda_error(self.ctx))
        return z, it, err

    def congruence(self, z, x, transpose_z=True):
        """Z^T X Z (transpose_z, Eq. 81) or Z X Z^T for symmetric x: one dmpt_congruence call."""
        t = self.torch
        if z.stride(0) != x.stride(0):
            raise DmptError(DMPT_EINVAL, "congruence", "z and x need the same leading dimension")
        c = t.empty((self.n, self.n), dtype=t.float32, device=self.device)
        rc = dmpt_congruence(self.ctx, z.data_ptr(), x.data_ptr(), z.stride(0), 1 if transpose_z else 0, c.data_ptr(),
                             self.n)
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_congruence", dmpt_last_cuda_error(self.ctx))
        return c

    def fd_response(self, h0, h1, n_occ, h, points=2, check=True):
        """(D1 by the 2- or 4-point stencil of PAPER.md Eqs. 83-84, layer counts of the runs, ms): order-0 contexts."""
        t = self.torch
        if h0.stride(0) != h1.stride(0):
            raise DmptError(DMPT_EINVAL, "fd_response", "h0 and h1 need the same leading dimension")
        d1 = t.empty((self.n, self.n), dtype=t.float32, device=self.device)
        rc, layers, ms = dmpt_fd_response(self.ctx, h0.data_ptr(), h1.data_ptr(), h0.stride(0), n_occ, h, points,
                                          d1.data_ptr(), self.n)
        if rc != DMPT_OK and check:
            raise DmptError(rc, "dmpt_fd_response", dmpt_last_cuda_error(self.ctx))
        return d1, layers, ms

    def spectral_bounds(self, h0):
        rc, lo, hi = dmpt_spectral_bounds(self.ctx, h0.data_ptr(), h0.stride(0))
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_spectral_bounds", dmpt_last_cuda_error(self.ctx))
        return lo, hi

    def initial_transform(self, h0, h1, eps_min, eps_max):
        t = self.torch
        s0 = t.empty((self.n, self.n), dtype=t.float32, device=self.device)
        s1 = t.empty((self.n, self.n), dtype=t.float32, device=self.device)
        rc, tr = dmpt_initial_transform(self.ctx, h0.data_ptr(), h1.data_ptr(), h0.stride(0), eps_min, eps_max,
                                        s0.data_ptr(), s1.data_ptr(), self.n)
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_initial_transform", dmpt_last_cuda_error(self.ctx))
        return s0, s1, tr

    def split(self, x, shift=0, diag_half=False):
        t = self.torch
        hi = t.empty((self.n, self.n), dtype=t.float16, device=self.device)
        lo = t.empty((self.n, self.n), dtype=t.float16, device=self.device)
        rc = dmpt_split(self.ctx, x.data_ptr(), x.stride(0), shift, 1 if diag_half else 0, hi.data_ptr(),
                        lo.data_ptr(), self.n)
        if rc != DMPT_OK:
            raise DmptError(rc, "dmpt_split", dmpt_last_cuda_error(self.ctx))
        return hi, lo

    def close(self):
        if getattr(self, "ctx", None) is not None:
            dmpt_destroy(self.ctx)
            self.ctx = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class DmptPair:
    """Order-parallel pair (dmpt_pair_*): the order-0 side on `device0`, the order-1 side on `device1` (the same
    device is allowed).  Owns both torch-allocated workspaces.  Marshalling only."""

    def __init__(self, n, device0="cuda:0", device1="cuda:0", max_layers=200, s0_shift=-1, s1_autoscale=True,
                 bounds=None, wave_sync=True, epilogue_direct=False, lanczos_steps=0):
        import torch

        self.torch = torch
        self.n = int(n)
        self.order = 1
        self.num_fields = 1
        self.dev = [torch.device(device0), torch.device(device1)]
        if any(d.type != "cuda" for d in self.dev):
            raise DmptError(DMPT_ECUDA, "DmptPair", "CUDA devices are required; there is no CPU path")
        opt = dmpt_default_options()
        opt.max_layers = min(int(max_layers) if int(max_layers) > 0 else 200, 1024)
        opt.order = 1
        opt.s0_shift = int(s0_shift)
        opt.s1_autoscale = 1 if s1_autoscale else 0
        opt.wave_sync = 1 if wave_sync else 0
        opt.epilogue_direct = 1 if epilogue_direct else 0
        if isinstance(bounds, str):
            opt.bounds = 2
            opt.lanczos_steps = int(lanczos_steps)
        elif bounds is not None:
            opt.bounds = 1
            opt.eps_min, opt.eps_max = float(bounds[0]), float(bounds[1])
        self.max_layers = opt.max_layers
        self.ws = []
        for side, d in enumerate(self.dev):
            nbytes = dmpt_pair_workspace_bytes(self.n, side)
            if nbytes == 0:
                raise DmptError(DMPT_EINVAL, "dmpt_pair_workspace_bytes")
            self.ws.append(torch.empty(nbytes, dtype=torch.uint8, device=d))
        idx = [d.index if d.index is not None else torch.cuda.current_device() for d in self.dev]
        self.pair = dmpt_pair_create(self.n, opt, idx[0], self.ws[0].data_ptr(), self.ws[0].numel(),
                                     idx[1], self.ws[1].data_ptr(), self.ws[1].numel())
        self._h = None

    _new_result = Dmpt._new_result
    _wrap_result = Dmpt._wrap

    def set_hamiltonian(self, h0, h1, n_occ):
        t = self.torch
        for m, d in ((h0, self.dev[0]), (h1, self.dev[1])):
            if not (m.is_cuda and m.dtype == t.float32 and m.dim() == 2 and m.stride(1) == 1
                    and m.stride(0) == h0.stride(0) and m.device.index == (d.index if d.index is not None else 0)):
                raise DmptError(DMPT_EINVAL, "DmptPair.set_hamiltonian",
                                "need row-major fp32 matrices, h0 on device0 and h1 on device1, one leading dimension")
        self._h = (h0, h1)
        dmpt_pair_set_hamiltonian(self.pair, h0.data_ptr(), h1.data_ptr(), h0.stride(0), n_occ)

    def run(self, check=True) -> DmptResult:
        t = self.torch
        n = self.n
        for d in self.dev:            # inputs may have been produced on torch's streams; the pair owns its own
            t.cuda.synchronize(d)
        d0 = t.empty((n, n), dtype=t.float32, device=self.dev[0])
        d1 = t.empty((n, n), dtype=t.float32, device=self.dev[1])
        r, bufs = self._new_result()
        rc = dmpt_pair_run(self.pair, d0.data_ptr(), d1.data_ptr(), n, r)
        if rc not in (DMPT_OK, DMPT_ENOCONV) and check:
            raise DmptError(rc, "dmpt_pair_run", dmpt_pair_last_cuda_error(self.pair))
        self.ctx = None
        return self._wrap_result(rc, r, bufs, d0, d1, None, False)

    def close(self):
        if getattr(self, "pair", None) is not None:
            dmpt_pair_destroy(self.pair)
            self.pair = None
            self.ws = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
