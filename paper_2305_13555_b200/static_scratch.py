"""Binding of include/oci_static.h: the library's one entry point that allocates nothing (its scratch memory is a
file-scope device array of 260 KiB inside liboci_b200.so; up to 1 048 576 cells).  Argument marshalling only."""
import ctypes as C

from .binding import OCIError, load_library

MAX_CELLS = 1048576
SCRATCH_BYTES = 256 + (MAX_CELLS // 64) * 16
SYMBOLS = ["oci_static_prepare", "oci_static_scalar_flux_norms", "oci_static_last_error"]

_ready = False


def _lib():
    global _ready
    L = load_library()
    if not _ready:
        vp = C.c_void_p
        L.oci_static_prepare.restype = C.c_int
        L.oci_static_prepare.argtypes = []
        L.oci_static_scalar_flux_norms.restype = C.c_int
        L.oci_static_scalar_flux_norms.argtypes = [vp, vp, vp, vp, vp, C.c_int64, C.c_int32, vp]
        L.oci_static_last_error.restype = C.c_char_p
        L.oci_static_last_error.argtypes = []
        _ready = True
    return L


def _check(L, rc):
    if rc != 0:
        raise OCIError(rc, L.oci_static_last_error().decode())


def static_prepare():
    """Once per device, with that device current (and before any stream capture)."""
    L = _lib()
    _check(L, L.oci_static_prepare())


def static_scalar_flux_norms(psi, w, phi_old, phi, norms, cells=None, n_angles=None, stream=None):
    """psi [cells][n_angles][4], w [n_angles], phi_old [cells][4] or None, phi [cells][4] (out), norms [2] (out): float64
    CUDA tensors on the current device.  `cells` / `n_angles` default to psi's shape.  Runs on `stream` (a raw
    cudaStream_t as an int) or on torch's current stream."""
    import torch
    L = _lib()
    cells = int(psi.shape[0]) if cells is None else int(cells)
    n_angles = int(psi.shape[1]) if n_angles is None else int(n_angles)
    for t in (psi, w, phi, norms) + (() if phi_old is None else (phi_old,)):
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    rc = L.oci_static_scalar_flux_norms(C.c_void_p(psi.data_ptr()), C.c_void_p(w.data_ptr()),
                                        C.c_void_p(phi_old.data_ptr()) if phi_old is not None else None,
                                        C.c_void_p(phi.data_ptr()), C.c_void_p(norms.data_ptr()), cells, n_angles, C.c_void_p(stream))
    _check(L, rc)
