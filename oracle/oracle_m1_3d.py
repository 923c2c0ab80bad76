"""ctypes wrapper around oracle/oracle_m1_3d.c — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle_m1.py)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_m1_3d.c")
_LIB = os.path.join(_HERE, "liboracle_m1_3d.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fvisibility=hidden", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"],
                       check=True, capture_output=True, text=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.oracle3_create.restype = C.c_void_p
        L.oracle3_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, ip]
        L.oracle3_destroy.argtypes = [C.c_void_p]
        L.oracle3_set_state.argtypes = [C.c_void_p, dp, dp, dp, dp]
        L.oracle3_get_state.argtypes = [C.c_void_p, dp, dp]
        L.oracle3_step_explicit.argtypes = [C.c_void_p, C.c_double]
        L.oracle3_step_implicit.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, dp]
        L.oracle3_residual.argtypes = [C.c_void_p, dp]
        L.oracle3_apply_linear.argtypes = [C.c_void_p, C.c_double, dp, dp]
        L.oracle3_diag_blocks.argtypes = [C.c_void_p, C.c_double, dp]
        L.oracle3_closure_point.argtypes = [C.c_double, C.c_double, dp, dp]
        L.oracle3_closure_point.restype = None
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a, shape):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.shape != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


class OracleM1_3D:
    """Arrays are [nz, ny, nx]; F is [3, nz, ny, nx].  bc = (xlo, xhi, ylo, yhi, zlo, zhi) with 0 periodic, 2 outflow."""

    def __init__(self, nx, ny, nz, dx, dy, dz, c=1.0, bc=(0, 0, 0, 0, 0, 0)):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        b = (C.c_int * 6)(*[int(v) for v in bc])
        self._h = lib().oracle3_create(self.nx, self.ny, self.nz, float(dx), float(dy), float(dz), float(c), b)
        if not self._h:
            raise ValueError("oracle3_create failed (bad arguments)")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().oracle3_destroy(self._h)
            self._h = None

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    def set_state(self, E, F, sigma_a, sigma_s):
        s = self.shape
        E, F, sa, ss = _f64(E, s), _f64(F, (3,) + s), _f64(sigma_a, s), _f64(sigma_s, s)
        lib().oracle3_set_state(self._h, _p(E), _p(F), _p(sa), _p(ss))

    def get_state(self):
        E, F = np.empty(self.shape), np.empty((3,) + self.shape)
        lib().oracle3_get_state(self._h, _p(E), _p(F))
        return E, F

    def step_explicit(self, dt):
        if lib().oracle3_step_explicit(self._h, float(dt)) < 0:
            raise RuntimeError("oracle3_step_explicit failed")

    def step_implicit(self, dt, tol=1e-10, restart=30, maxit=4000):
        res = C.c_double(0.0)
        its = lib().oracle3_step_implicit(self._h, float(dt), float(tol), int(restart), int(maxit), C.byref(res))
        if its < 0:
            raise RuntimeError("oracle3_step_implicit failed")
        return its, res.value

    def residual(self):
        R = np.empty((4,) + self.shape)
        lib().oracle3_residual(self._h, _p(R))
        return R

    def apply_linear(self, dt, V):
        V = _f64(V, (4,) + self.shape)
        out = np.empty_like(V)
        lib().oracle3_apply_linear(self._h, float(dt), _p(V), _p(out))
        return out

    def diag_blocks(self, dt):
        B = np.empty((self.nx * self.ny * self.nz, 4, 4))
        lib().oracle3_diag_blocks(self._h, float(dt), _p(B))
        return B


def closure_point(c, E, F):
    F = np.ascontiguousarray(F, dtype=np.float64)
    out = np.empty(52)
    lib().oracle3_closure_point(float(c), float(E), _p(F), _p(out))
    return dict(f=out[0], P=out[1:10].reshape(3, 3).copy(), lmin=out[10:13].copy(), lmax=out[13:16].copy(), J=out[16:52].reshape(3, 3, 4).copy())
