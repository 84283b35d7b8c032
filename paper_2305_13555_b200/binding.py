"""ctypes binding with the same names as include/oci.h."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

BC_VACUUM, BC_INCIDENT_ISOTROPIC, BC_REFLECTING, BC_HALO = 0, 1, 2, 3
PATH_SHARED, PATH_PER_CELL = 0, 1
KERNEL_GENERIC, KERNEL_RESIDENT, KERNEL_KTILED, KERNEL_PER_CELL = 0, 1, 2, 3
ITERATION_FULL, ITERATION_REDUCED, ITERATION_AUTO = 0, 1, 2
RKERNEL_AUTO, RKERNEL_GEMV, RKERNEL_RESIDENT, RKERNEL_KTILED, RKERNEL_OPREG, RKERNEL_WOODBURY = -1, 0, 1, 2, 3, 4

EXPORTED_SYMBOLS = [
    "oci_create", "oci_workspace_bytes", "oci_setup", "oci_set_flux", "oci_set_flux_dev", "oci_set_source",
    "oci_set_source_dev", "oci_step", "si_step", "oci_get_scalar_flux", "oci_get_angular_flux",
    "oci_get_scalar_flux_dev", "oci_get_angular_flux_dev", "oci_get_scalar_flux_async", "oci_synchronize", "oci_get_quadrature", "oci_get_info",
    "oci_get_block_inverse", "oci_enable_kernel_timing", "oci_get_kernel_time", "oci_get_aux_kernel_time", "oci_set_iteration", "oci_set_reduced_kernel", "oci_set_small_step", "oci_get_setup_time", "oci_shard_mailbox_bytes", "oci_shard_attach", "oci_shard_step", "oci_launch_count",
    "oci_last_error", "oci_destroy",
]


class OCIError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"oci error {code}: {msg}")
        self.code = code


class _bc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("value", C.c_double)]


class _info(C.Structure):
    _fields_ = [("cells", C.c_int64), ("n_angles", C.c_int32), ("block_dim", C.c_int32),
                ("n_blocks", C.c_int64), ("path", C.c_int32), ("apply_kernel", C.c_int32),
                ("iteration", C.c_int32), ("reduced_kernel", C.c_int32), ("small_step_cluster", C.c_int32),
                ("si_small_step_cluster", C.c_int32)]


_dp = C.POINTER(C.c_double)
_lib = None


def library_path() -> str:
    return _build.LIB


def load_library():
    """Load liboci_b200.so (building it with nvcc if it is missing or stale).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    if not os.path.exists(path):
        raise OCIError(-3, f"CUDA library {path} is missing and could not be built")
    L = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.oci_create.restype = C.c_int
    L.oci_create.argtypes = [C.POINTER(vp), i64, _dp, _dp, _dp, dbl, dbl, i32, _bc, _bc]
    L.oci_workspace_bytes.restype = i64
    L.oci_workspace_bytes.argtypes = [vp]
    L.oci_setup.restype = C.c_int
    L.oci_setup.argtypes = [vp, vp, i64, vp]
    for name in ("oci_set_flux", "oci_set_source", "oci_get_scalar_flux", "oci_get_angular_flux"):
        f = getattr(L, name)
        f.restype = C.c_int
        f.argtypes = [vp, _dp]
    for name in ("oci_set_flux_dev", "oci_set_source_dev", "oci_get_scalar_flux_dev", "oci_get_angular_flux_dev"):
        f = getattr(L, name)
        f.restype = C.c_int
        f.argtypes = [vp, vp]
    for name in ("oci_step", "si_step"):
        f = getattr(L, name)
        f.restype = C.c_int
        f.argtypes = [vp, dbl, i32, C.POINTER(i32), _dp]
    L.oci_get_scalar_flux_async.restype = C.c_int
    L.oci_get_scalar_flux_async.argtypes = [vp, vp]
    L.oci_synchronize.restype = C.c_int
    L.oci_synchronize.argtypes = [vp]
    L.oci_get_quadrature.restype = C.c_int
    L.oci_get_quadrature.argtypes = [vp, _dp, _dp]
    L.oci_get_info.restype = C.c_int
    L.oci_get_info.argtypes = [vp, C.POINTER(_info)]
    L.oci_get_block_inverse.restype = C.c_int
    L.oci_get_block_inverse.argtypes = [vp, i64, _dp]
    L.oci_enable_kernel_timing.restype = C.c_int
    L.oci_enable_kernel_timing.argtypes = [vp, i32]
    L.oci_get_kernel_time.restype = C.c_int
    L.oci_get_kernel_time.argtypes = [vp, _dp, C.POINTER(i64)]
    L.oci_get_aux_kernel_time.restype = C.c_int
    L.oci_get_aux_kernel_time.argtypes = [vp, _dp, C.POINTER(i64), _dp, C.POINTER(i64)]
    L.oci_set_iteration.restype = C.c_int
    L.oci_set_iteration.argtypes = [vp, i32]
    L.oci_set_reduced_kernel.restype = C.c_int
    L.oci_set_reduced_kernel.argtypes = [vp, i32]
    L.oci_set_small_step.restype = C.c_int
    L.oci_set_small_step.argtypes = [vp, i32]
    L.oci_get_setup_time.restype = C.c_int
    L.oci_get_setup_time.argtypes = [vp, _dp]
    L.oci_shard_mailbox_bytes.restype = i64
    L.oci_shard_mailbox_bytes.argtypes = [i32, i32]
    L.oci_shard_attach.restype = C.c_int
    L.oci_shard_attach.argtypes = [vp, i32, i32, C.POINTER(vp)]
    L.oci_shard_step.restype = C.c_int
    L.oci_shard_step.argtypes = [C.POINTER(vp), i32, dbl, i32, C.POINTER(i32), _dp]
    L.oci_launch_count.restype = i64
    L.oci_launch_count.argtypes = [vp]
    L.oci_last_error.restype = C.c_char_p
    L.oci_last_error.argtypes = [vp]
    L.oci_destroy.restype = None
    L.oci_destroy.argtypes = [vp]
    _lib = L
    return L


def _hp(a):
    return a.ctypes.data_as(_dp)


_probe = None


def probe_fp64_tensor_tflops(device="cuda:0") -> float:
    """fp64 tensor-pipe (DMMA) issue rate of `device` in TFLOP/s, from the measurement probe liboci_probe.so
    (not part of the product ABI), on torch's current stream."""
    import torch
    global _probe
    if _probe is None:
        _build.build()
        _probe = C.CDLL(_build.PROBE_LIB)
        _probe.oci_probe_fp64_tensor_tflops.restype = C.c_int
        _probe.oci_probe_fp64_tensor_tflops.argtypes = [C.c_void_p, C.c_void_p, _dp]
    L = _probe
    dev = torch.device(device)
    with torch.cuda.device(dev):
        scratch = torch.zeros(8, dtype=torch.float64, device=dev)
        out = C.c_double(0.0)
        rc = L.oci_probe_fp64_tensor_tflops(C.c_void_p(scratch.data_ptr()),
                                            C.c_void_p(torch.cuda.current_stream(dev).cuda_stream), C.byref(out))
        if rc != 0:
            raise OCIError(rc, "oci_probe_fp64_tensor_tflops failed")
    return out.value


class OCI:
    """One problem on one GPU.  Method names follow include/oci.h."""

    def __init__(self, dx, sigma_t, sigma_s, v, dt, n_angles, bc_left=(BC_VACUUM, 0.0), bc_right=(BC_VACUUM, 0.0)):
        self._L = load_library()
        self._h = C.c_void_p()
        dx = np.ascontiguousarray(dx, dtype=np.float64)
        st = np.ascontiguousarray(sigma_t, dtype=np.float64)
        ss = np.ascontiguousarray(sigma_s, dtype=np.float64)
        if not (dx.ndim == 1 and dx.shape == st.shape == ss.shape):
            raise OCIError(-1, "dx, sigma_t, sigma_s must be 1-D arrays of equal length")
        rc = self._L.oci_create(C.byref(self._h), len(dx), _hp(dx), _hp(st), _hp(ss), float(v), float(dt),
                                int(n_angles), _bc(int(bc_left[0]), float(bc_left[1])),
                                _bc(int(bc_right[0]), float(bc_right[1])))
        if rc != 0:
            self._h = C.c_void_p()
            raise OCIError(rc, "oci_create: invalid argument")
        self.cells, self.n_angles = len(dx), int(n_angles)
        self._ws = None

    @classmethod
    def from_problem(cls, p, device="cuda:0", set_flux=True, iteration=None, reduced_kernel=None, small_step=None):
        o = cls(p.dx, p.sigma_t, p.sigma_s, p.v, p.dt, p.n_angles, p.bc_left, p.bc_right)
        if iteration is not None:
            o.set_iteration(iteration)
        if reduced_kernel is not None:
            o.set_reduced_kernel(reduced_kernel)
        if small_step is not None:
            o.set_small_step(small_step)
        o.setup(device)
        if set_flux:
            o.set_flux(p.psi0)
        return o

    # -- helpers
    def _check(self, rc, allow_not_converged=False):
        if rc < 0 or (rc == 1 and not allow_not_converged):
            raise OCIError(rc, self._L.oci_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None) and self._h:
            self._L.oci_destroy(self._h)
            self._h = C.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C ABI, one method per entry point
    def workspace_bytes(self) -> int:
        return int(self._L.oci_workspace_bytes(self._h))

    def setup(self, device="cuda:0", stream=None):
        """Allocates the workspace as a torch tensor on `device` and calls oci_setup on torch's
        current stream (or `stream`)."""
        import torch
        if not torch.cuda.is_available():
            raise OCIError(-3, "no CUDA device: this library has no CPU fallback")
        dev = torch.device(device)
        with torch.cuda.device(dev):
            self._ws = torch.empty(self.workspace_bytes() + 256, dtype=torch.uint8, device=dev)
            ptr = (self._ws.data_ptr() + 255) & ~255
            st = stream if stream is not None else torch.cuda.current_stream(dev)
            self._stream = st
            self._device = dev
            self._check(self._L.oci_setup(self._h, C.c_void_p(ptr), self.workspace_bytes(), C.c_void_p(st.cuda_stream)))
        return self

    def set_flux(self, psi_edge):
        a = np.ascontiguousarray(psi_edge, dtype=np.float64)
        if a.shape != (self.cells, self.n_angles, 2):
            raise OCIError(-1, "psi_edge must be [cells][N][2]")
        self._check(self._L.oci_set_flux(self._h, _hp(a)))

    def set_flux_dev(self, t):
        self._check(self._L.oci_set_flux_dev(self._h, C.c_void_p(t.data_ptr())))

    def set_source(self, q):
        if q is None:
            self._check(self._L.oci_set_source(self._h, None))
            return
        a = np.ascontiguousarray(q, dtype=np.float64)
        if a.shape != (self.cells, 4):
            raise OCIError(-1, "q must be [cells][4]")
        self._check(self._L.oci_set_source(self._h, _hp(a)))

    def set_source_dev(self, t):
        self._check(self._L.oci_set_source_dev(self._h, C.c_void_p(t.data_ptr()) if t is not None else None))

    def _step(self, f, tol, max_iters):
        out = self.__dict__.get("_step_out")             # the two out-parameters, made once (a small step is ~40 us in all)
        if out is None:
            it, res = C.c_int32(0), C.c_double(0.0)
            out = self.__dict__["_step_out"] = (it, res, C.byref(it), C.byref(res))
        rc = f(self._h, tol, max_iters, out[2], out[3])
        if rc < 0:
            self._check(rc, allow_not_converged=True)
        return rc, out[0].value, out[1].value

    def oci_step(self, tol=1e-10, max_iters=10_000):
        return self._step(self._L.oci_step, tol, max_iters)

    def si_step(self, tol=1e-10, max_iters=10_000):
        return self._step(self._L.si_step, tol, max_iters)

    def get_scalar_flux(self, out=None):
        a = np.empty((self.cells, 4)) if out is None else out
        assert a.dtype == np.float64 and a.flags.c_contiguous and a.shape == (self.cells, 4)
        self._check(self._L.oci_get_scalar_flux(self._h, _hp(a)))
        return a

    def get_scalar_flux_async(self, pinned):
        """`pinned`: a page-locked torch tensor [cells][4] float64 (torch.empty(...).pin_memory()); valid after synchronize()."""
        assert pinned.is_pinned() and pinned.dtype.itemsize == 8 and pinned.numel() == self.cells * 4 and pinned.is_contiguous()
        self._check(self._L.oci_get_scalar_flux_async(self._h, C.c_void_p(pinned.data_ptr())))

    def synchronize(self):
        self._check(self._L.oci_synchronize(self._h))

    def get_angular_flux(self):
        a = np.empty((self.cells, self.n_angles, 4))
        self._check(self._L.oci_get_angular_flux(self._h, _hp(a)))
        return a

    def get_scalar_flux_dev(self, t):
        self._check(self._L.oci_get_scalar_flux_dev(self._h, C.c_void_p(t.data_ptr())))

    def get_angular_flux_dev(self, t):
        self._check(self._L.oci_get_angular_flux_dev(self._h, C.c_void_p(t.data_ptr())))

    def get_quadrature(self):
        mu, w = np.empty(self.n_angles), np.empty(self.n_angles)
        self._check(self._L.oci_get_quadrature(self._h, _hp(mu), _hp(w)))
        return mu, w

    def get_info(self):
        i = _info()
        self._check(self._L.oci_get_info(self._h, C.byref(i)))
        return dict(cells=i.cells, n_angles=i.n_angles, block_dim=i.block_dim, n_blocks=i.n_blocks, path=i.path,
                    apply_kernel=i.apply_kernel, iteration=i.iteration, reduced_kernel=i.reduced_kernel,
                    small_step_cluster=i.small_step_cluster,
                    si_small_step_cluster=i.si_small_step_cluster)

    def get_block_inverse(self, blk=0):
        n = 4 * self.n_angles
        a = np.empty((n, n))
        self._check(self._L.oci_get_block_inverse(self._h, int(blk), _hp(a)))
        return a

    def enable_kernel_timing(self, on=True):
        self._check(self._L.oci_enable_kernel_timing(self._h, 1 if on else 0))

    def get_kernel_time(self):
        ms, k = C.c_double(0.0), C.c_int64(0)
        self._check(self._L.oci_get_kernel_time(self._h, C.byref(ms), C.byref(k)))
        return ms.value, k.value

    def get_aux_kernel_time(self):
        a, b, ka, kb = C.c_double(0.0), C.c_double(0.0), C.c_int64(0), C.c_int64(0)
        self._check(self._L.oci_get_aux_kernel_time(self._h, C.byref(a), C.byref(ka), C.byref(b), C.byref(kb)))
        return dict(fix_ms=a.value, fix_launches=ka.value, final_ms=b.value, final_launches=kb.value)

    def set_iteration(self, iteration):
        self._check(self._L.oci_set_iteration(self._h, int(iteration)))

    def set_reduced_kernel(self, kernel):
        self._check(self._L.oci_set_reduced_kernel(self._h, int(kernel)))

    def set_small_step(self, mode):
        self._check(self._L.oci_set_small_step(self._h, int(mode)))

    def shard_attach(self, rank, world, mailbox_ptrs):
        """oci_shard_attach: `mailbox_ptrs` = the W device addresses (ints) of all ranks' mailboxes, in rank order."""
        arr = (C.c_void_p * int(world))(*[C.c_void_p(int(p)) for p in mailbox_ptrs])
        self._check(self._L.oci_shard_attach(self._h, int(rank), int(world), arr))

    def get_setup_time(self) -> float:
        ms = C.c_double(0.0)
        self._check(self._L.oci_get_setup_time(self._h, C.byref(ms)))
        return ms.value

    def launch_count(self):
        return int(self._L.oci_launch_count(self._h))


def shard_mailbox_bytes(n_angles, world) -> int:
    return int(load_library().oci_shard_mailbox_bytes(int(n_angles), int(world)))


def shard_step(shards, tol=1e-10, max_iters=10_000):
    """oci_shard_step over the shards of one slab that live in this process (a list of OCI objects)."""
    L = load_library()
    arr = (C.c_void_p * len(shards))(*[s._h for s in shards])
    it, res = C.c_int32(0), C.c_double(0.0)
    rc = L.oci_shard_step(arr, len(shards), float(tol), int(max_iters), C.byref(it), C.byref(res))
    if rc < 0:
        raise OCIError(rc, L.oci_last_error(shards[0]._h).decode())
    return rc, it.value, res.value
