"""ctypes wrapper around oracle/oracle_m1.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It never imports the CUDA package, and the CUDA package never imports it.

The arithmetic lives in oracle_m1.c (see its header for the PAPER.md passages it follows); this file only
builds the shared object with gcc and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_m1.c")
_LIB = os.path.join(_HERE, "liboracle_m1.so")

BC_PERIODIC, BC_DIRICHLET, BC_OUTFLOW = 0, 1, 2
XLO, XHI, YLO, YHI = 0, 1, 2, 3

_lib = None


def build(force: bool = False) -> str:
    """Compile oracle_m1.c -> liboracle_m1.so (gcc -O2, OpenMP, no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fvisibility=hidden", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True, text=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip, lp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_long)
        L.oracle_m1_create.restype = C.c_void_p
        L.oracle_m1_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, ip]
        L.oracle_m1_destroy.argtypes = [C.c_void_p]
        L.oracle_m1_set_state.argtypes = [C.c_void_p, dp, dp, dp, dp, dp]
        L.oracle_m1_set_boundary.argtypes = [C.c_void_p, C.c_int, dp, dp, dp, dp]
        L.oracle_m1_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_double]
        L.oracle_m1_set_field.argtypes = [C.c_void_p, C.c_char_p, dp]
        L.oracle_m1_get_state.argtypes = [C.c_void_p, dp, dp, dp]
        L.oracle_m1_step_explicit.argtypes = [C.c_void_p, C.c_double]
        L.oracle_m1_step_implicit.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, dp]
        L.oracle_m1_step_semi_implicit.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, dp]
        L.oracle_m1_step_implicit_newton.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, C.c_int, ip, dp, dp]
        L.oracle_m1_add_velocity_sources.argtypes = [C.c_void_p, C.c_double]
        L.oracle_m1_residual.argtypes = [C.c_void_p, dp, dp]
        L.oracle_m1_apply_linear.argtypes = [C.c_void_p, C.c_double, dp, dp, C.c_int]
        L.oracle_m1_assemble.argtypes = [C.c_void_p, C.c_double, dp, lp, dp]
        L.oracle_m1_count_unrealizable.argtypes = [C.c_void_p, lp, lp]
        L.oracle_m1_mg_apply.argtypes = [C.c_void_p, C.c_double, dp, dp]
        L.oracle_m1_mg_level.argtypes = [C.c_void_p, C.c_double, C.c_int, dp, lp, ip]
        L.oracle_m1_get_history.argtypes = [C.c_void_p, dp, C.c_int]
        L.oracle_m1_last_error.restype = C.c_char_p
        L.oracle_m1_last_error.argtypes = [C.c_void_p]
        L.oracle_m1_closure_point.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, dp]
        L.oracle_m1_face_point.argtypes = [C.c_void_p, dp, dp, C.c_int, dp]
        L.oracle_m1_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None and a.shape != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


class OracleM1:
    """Same calls as the CUDA binding (paper_2011_13926_b200.ArkM1), host numpy arrays."""

    def __init__(self, nx, ny, dx, dy, c=1.0, bc=(0, 0, 0, 0)):
        self.nx, self.ny, self.dx, self.dy, self.c = int(nx), int(ny), float(dx), float(dy), float(c)
        bc_arr = (C.c_int * 4)(*[int(b) for b in bc])
        self._h = lib().oracle_m1_create(self.nx, self.ny, self.dx, self.dy, self.c, bc_arr)
        if not self._h:
            raise ValueError("oracle_m1_create failed (bad arguments)")
        self.bc = tuple(int(b) for b in bc)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().oracle_m1_destroy(self._h)
            self._h = None

    def _check(self, rc):
        if rc < 0:
            raise RuntimeError(lib().oracle_m1_last_error(self._h).decode())
        return rc

    @property
    def shape(self):
        return (self.ny, self.nx)

    def set_state(self, E, F, sigma_a, sigma_s, T=None):
        s = self.shape
        E, F = _f64(E, s), _f64(F, (2,) + s)
        sa, ss = _f64(sigma_a, s), _f64(sigma_s, s)
        T = None if T is None else _f64(T, s)
        self._check(lib().oracle_m1_set_state(self._h, _p(E), _p(F), _p(sa), _p(ss), _p(T)))

    def set_boundary(self, side, E_g, F_g, sigma_a_g, sigma_s_g):
        n = self.ny if side < 2 else self.nx
        E_g, F_g = _f64(E_g, (n,)), _f64(F_g, (2, n))
        sa, ss = _f64(sigma_a_g, (n,)), _f64(sigma_s_g, (n,))
        self._check(lib().oracle_m1_set_boundary(self._h, side, _p(E_g), _p(F_g), _p(sa), _p(ss)))

    def set_option(self, key, value):
        self._check(lib().oracle_m1_set_option(self._h, key.encode(), float(value)))

    def set_field(self, name, plane):
        plane = None if plane is None else _f64(plane, self.shape)
        self._check(lib().oracle_m1_set_field(self._h, name.encode(), _p(plane)))

    def get_state(self, with_T=False):
        E = np.empty(self.shape)
        F = np.empty((2,) + self.shape)
        T = np.empty(self.shape) if with_T else None
        self._check(lib().oracle_m1_get_state(self._h, _p(E), _p(F), _p(T)))
        return (E, F, T) if with_T else (E, F)

    def step_explicit(self, dt):
        self._check(lib().oracle_m1_step_explicit(self._h, float(dt)))

    def step_implicit(self, dt, tol=1e-10, restart=30, maxit=4000):
        res = C.c_double(0.0)
        its = self._check(lib().oracle_m1_step_implicit(self._h, float(dt), float(tol), int(restart), int(maxit), C.byref(res)))
        return its, res.value

    def step_semi_implicit(self, dt, tol=1e-12, restart=30, maxit=4000):
        res = C.c_double(0.0)
        its = self._check(lib().oracle_m1_step_semi_implicit(self._h, float(dt), float(tol), int(restart), int(maxit), C.byref(res)))
        return its, res.value

    def step_implicit_newton(self, dt, tol=1e-10, restart=30, maxit=4000, newton_tol=1e-8, max_newton=20):
        """Returns (total GMRES iterations, Newton iterations, last true relative residual, last relative update)."""
        nn, res, upd = C.c_int(0), C.c_double(0.0), C.c_double(0.0)
        its = self._check(lib().oracle_m1_step_implicit_newton(self._h, float(dt), float(tol), int(restart), int(maxit), float(newton_tol),
                                                               int(max_newton), C.byref(nn), C.byref(res), C.byref(upd)))
        return its, nn.value, res.value, upd.value

    def add_velocity_sources(self, dt):
        self._check(lib().oracle_m1_add_velocity_sources(self._h, float(dt)))

    # ---- test hooks -------------------------------------------------------------------------------
    def residual(self):
        RE = np.empty(self.shape)
        RF = np.empty((2,) + self.shape)
        self._check(lib().oracle_m1_residual(self._h, _p(RE), _p(RF)))
        return RE, RF

    def apply_linear(self, dt, V, mode=0):
        V = _f64(V, (3,) + self.shape)
        out = np.empty_like(V)
        self._check(lib().oracle_m1_apply_linear(self._h, float(dt), _p(V), _p(out), int(mode)))
        return out

    def assemble(self, dt):
        """Returns A[N,5,3,3] (centre, west, east, south, north), col[N,5] (cell index or -1), b[3,ny,nx]."""
        N = self.nx * self.ny
        A = np.empty((N, 5, 3, 3))
        col = np.empty((N, 5), dtype=np.int64)
        b = np.empty((3,) + self.shape)
        self._check(lib().oracle_m1_assemble(self._h, float(dt), _p(A), col.ctypes.data_as(C.POINTER(C.c_long)), _p(b)))
        return A, col, b

    def dense_matrix(self, dt):
        """Dense (3N x 3N) matrix in plane ordering [E | Fx | Fy] and b (3N), from the assembled blocks."""
        A, col, b = self.assemble(dt)
        N = self.nx * self.ny
        M = np.zeros((3 * N, 3 * N))
        for cell in range(N):
            for k in range(5):
                cj = col[cell, k]
                if cj < 0:
                    continue
                for r in range(3):
                    for s in range(3):
                        M[r * N + cell, s * N + cj] += A[cell, k, r, s]
        return M, b.reshape(-1)

    def mg_apply(self, dt, R):
        """One multigrid V-cycle z = M^-1 r on the system assembled for dt (planes [3, ny, nx])."""
        R = _f64(R, (3,) + self.shape)
        out = np.empty_like(R)
        self._check(lib().oracle_m1_mg_apply(self._h, float(dt), _p(R), _p(out)))
        return out

    def mg_level(self, dt, level):
        """(number of levels, nx_l, ny_l, A[N_l,5,3,3], col[N_l,5]) of one level of the multigrid hierarchy."""
        dims = (C.c_int * 2)()
        n = lib().oracle_m1_mg_level(self._h, float(dt), int(level), None, None, dims)
        self._check(min(n, 0))
        nx, ny = dims[0], dims[1]
        A = np.empty((nx * ny, 5, 3, 3)); col = np.empty((nx * ny, 5), dtype=np.int64)
        lib().oracle_m1_mg_level(self._h, float(dt), int(level), _p(A), col.ctypes.data_as(C.POINTER(C.c_long)), dims)
        return n, nx, ny, A, col

    def count_unrealizable(self):
        a, b = C.c_long(0), C.c_long(0)
        self._check(lib().oracle_m1_count_unrealizable(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def history(self):
        n = lib().oracle_m1_get_history(self._h, None, 0)
        buf = np.empty(max(n, 1))
        lib().oracle_m1_get_history(self._h, _p(buf), n)
        return buf[:n]

    def closure_point(self, E, Fx, Fy):
        out = np.empty(21)
        lib().oracle_m1_closure_point(self._h, float(E), float(Fx), float(Fy), _p(out))
        return dict(f=out[0], fx=out[1], fy=out[2], xi=out[3], chi=out[4], Pxx=out[5], Pxy=out[6], Pyy=out[7],
                    lmin_x=out[8], lmax_x=out[9], lmin_y=out[10], lmax_y=out[11], J=out[12:21].reshape(3, 3).copy())

    def face_point(self, UL, UR, direction):
        """UL, UR = (E, Fx, Fy, sigma_a, sigma_t). Returns a+, a-, Lambda, alpha, sigma_f."""
        UL, UR = _f64(UL, (5,)), _f64(UR, (5,))
        out = np.empty(5)
        lib().oracle_m1_face_point(self._h, _p(UL), _p(UR), int(direction), _p(out))
        return dict(ap=out[0], am=out[1], Lam=out[2], alpha=out[3], sig=out[4])


def num_threads():
    return lib().oracle_m1_num_threads()
