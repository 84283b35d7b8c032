"""ctypes loader for oracle/mbscb_oracle.c (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def _p(a):
    return a.ctypes.data_as(_dp)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_double, C.c_double, C.c_int32,
                                 C.c_int32, C.c_double, C.c_int32, C.c_double]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int32]
        L.orc_threads_available.restype = C.c_int32
        L.orc_setup.restype = C.c_int64
        L.orc_setup.argtypes = [C.c_void_p]
        L.orc_set_flux.argtypes = [C.c_void_p, _dp]
        L.orc_set_source.argtypes = [C.c_void_p, _dp]
        L.orc_set_iterate.argtypes = [C.c_void_p, _dp]
        for f in (L.orc_oci_iteration, L.orc_si_iteration):
            f.argtypes = [C.c_void_p, _dp, _dp]
        for f in (L.orc_oci_step, L.orc_si_step):
            f.restype = C.c_int32
            f.argtypes = [C.c_void_p, C.c_double, C.c_int32, _ip, _dp]
        L.orc_get_scalar_flux.argtypes = [C.c_void_p, _dp]
        L.orc_get_angular_flux.argtypes = [C.c_void_p, _dp]
        L.orc_get_prev_edge_flux.argtypes = [C.c_void_p, _dp]
        L.orc_get_quadrature.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_num_blocks.restype = C.c_int64
        L.orc_num_blocks.argtypes = [C.c_void_p]
        L.orc_gauss_legendre.argtypes = [C.c_int32, _dp, _dp]
        L.orc_A4.argtypes = [C.c_double] * 5 + [_dp]
        L.orc_cell_matrix.argtypes = [C.c_int32, _dp, _dp, C.c_double, C.c_double, C.c_double,
                                      C.c_double, C.c_double, _dp]
        L.orc_lu_factor.restype = C.c_int32
        L.orc_lu_factor.argtypes = [C.c_int32, _dp, _ip]
        L.orc_lu_solve.argtypes = [C.c_int32, _dp, _ip, _dp]
        _lib = L
    return _lib


def threads_available() -> int:
    return int(lib().orc_threads_available())


def gauss_legendre(N: int):
    mu = np.empty(N)
    w = np.empty(N)
    lib().orc_gauss_legendre(N, _p(mu), _p(w))
    return mu, w


def A4(mu, dx, sig, v, dt):
    A = np.empty((4, 4))
    lib().orc_A4(mu, dx, sig, v, dt, _p(A))
    return A


def cell_matrix(mu, w, dx, sig, sigs, v, dt):
    mu = np.ascontiguousarray(mu, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    N = len(mu)
    B = np.empty((4 * N, 4 * N))
    lib().orc_cell_matrix(N, _p(mu), _p(w), dx, sig, sigs, v, dt, _p(B))
    return B


def lu_factor(A):
    LU = np.array(A, dtype=np.float64, order="C")
    n = LU.shape[0]
    piv = np.empty(n, dtype=np.int32)
    info = lib().orc_lu_factor(n, _p(LU), piv.ctypes.data_as(_ip))
    return LU, piv, int(info)


def lu_solve(LU, piv, b):
    x = np.array(b, dtype=np.float64, order="C")
    lib().orc_lu_solve(LU.shape[0], _p(LU), piv.ctypes.data_as(_ip), _p(x))
    return x


class Oracle:
    """One MB-SCB problem on the CPU oracle.  Mirrors the problem statement of
    PAPER.md:49-61 (cells, dx, Sigma, Sigma_s, v, dt, quadrature order, BCs)."""

    def __init__(self, dx, sigma_t, sigma_s, v, dt, n_angles, bc_left=(0, 0.0), bc_right=(0, 0.0),
                 threads: int = 1):
        self.dx = np.ascontiguousarray(dx, dtype=np.float64)
        self.sigma_t = np.ascontiguousarray(sigma_t, dtype=np.float64)
        self.sigma_s = np.ascontiguousarray(sigma_s, dtype=np.float64)
        self.J = len(self.dx)
        self.N = int(n_angles)
        self.n = 4 * self.N
        self.v, self.dt = float(v), float(dt)
        self._h = lib().orc_create(self.J, _p(self.dx), _p(self.sigma_t), _p(self.sigma_s), self.v,
                                   self.dt, self.N, int(bc_left[0]), float(bc_left[1]),
                                   int(bc_right[0]), float(bc_right[1]))
        if not self._h:
            raise ValueError("oracle: invalid problem")
        lib().orc_set_threads(self._h, int(threads))
        self.threads = int(threads)

    @classmethod
    def from_problem(cls, p, threads: int = 1):
        o = cls(p.dx, p.sigma_t, p.sigma_s, p.v, p.dt, p.n_angles, p.bc_left, p.bc_right, threads)
        o.setup()
        o.set_flux(p.psi0)
        return o

    def __del__(self):
        try:
            if self._h:
                lib().orc_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def setup(self):
        bad = lib().orc_setup(self._h)
        if bad:
            raise np.linalg.LinAlgError(f"oracle: singular cell block {bad - 1}")

    @property
    def num_blocks(self):
        return int(lib().orc_num_blocks(self._h))

    def set_flux(self, psi_edge):
        a = np.ascontiguousarray(psi_edge, dtype=np.float64)
        assert a.shape == (self.J, self.N, 2)
        lib().orc_set_flux(self._h, _p(a))

    def set_source(self, q):
        if q is None:
            lib().orc_set_source(self._h, None)
        else:
            a = np.ascontiguousarray(q, dtype=np.float64)
            assert a.shape == (self.J, 4)
            lib().orc_set_source(self._h, _p(a))

    def set_iterate(self, psi):
        a = np.ascontiguousarray(psi, dtype=np.float64).reshape(self.J, self.n)
        lib().orc_set_iterate(self._h, _p(a))

    def _iter(self, f):
        d, r = C.c_double(), C.c_double()
        f(self._h, C.byref(d), C.byref(r))
        return d.value, r.value

    def oci_iteration(self):
        return self._iter(lib().orc_oci_iteration)

    def si_iteration(self):
        return self._iter(lib().orc_si_iteration)

    def _step(self, f, tol, max_iters):
        it, res = C.c_int32(), C.c_double()
        st = f(self._h, float(tol), int(max_iters), C.byref(it), C.byref(res))
        if st < 0:
            raise RuntimeError(f"oracle step failed: {st}")
        return st, it.value, res.value

    def oci_step(self, tol=1e-10, max_iters=10_000):
        return self._step(lib().orc_oci_step, tol, max_iters)

    def si_step(self, tol=1e-10, max_iters=10_000):
        return self._step(lib().orc_si_step, tol, max_iters)

    def scalar_flux(self):
        a = np.empty((self.J, 4))
        lib().orc_get_scalar_flux(self._h, _p(a))
        return a

    def angular_flux(self):
        a = np.empty((self.J, self.N, 4))
        lib().orc_get_angular_flux(self._h, _p(a))
        return a

    def prev_edge_flux(self):
        a = np.empty((self.J, self.N, 2))
        lib().orc_get_prev_edge_flux(self._h, _p(a))
        return a

    def quadrature(self):
        mu, w = np.empty(self.N), np.empty(self.N)
        lib().orc_get_quadrature(self._h, _p(mu), _p(w))
        return mu, w
