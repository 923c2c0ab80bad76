"""Thin ctypes binding of libark_m1.so (include/ark_m1.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/.  There is no CPU fallback: if the shared library is
missing or cannot be loaded this module raises.  torch is used only for device memory and streams; array
arguments may be torch tensors (cuda or cpu, float64, contiguous) or numpy float64 arrays — their raw pointers
are passed straight to the C ABI, which accepts host and device pointers alike.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libark_m1.so")

BC_PERIODIC, BC_DIRICHLET, BC_OUTFLOW = 0, 1, 2
XLO, XHI, YLO, YHI = 0, 1, 2, 3

# every symbol include/ark_m1.h declares
SYMBOLS = [
    "ark_m1_create", "ark_m1_destroy", "ark_m1_set_stream", "ark_m1_set_state", "ark_m1_set_boundary",
    "ark_m1_set_option", "ark_m1_set_field", "ark_m1_get_state", "ark_m1_prefetch_state", "ark_m1_commit_state", "ark_m1_get_state_async", "ark_m1_wait_transfers", "ark_m1_step_explicit", "ark_m1_steps_explicit",
    "ark_m1_step_implicit", "ark_m1_step_implicit_newton", "ark_m1_step_semi_implicit", "ark_m1_add_velocity_sources", "ark_m1_count_unrealizable", "ark_m1_residual",
    "ark_m1_apply_operator", "ark_m1_get_history", "ark_m1_get_timings", "ark_m1_get_kernel_stats",
    "ark_m1_kernel_class_name", "ark_m1_kernel_launches", "ark_m1_block_stats", "ark_m1_fastmath_errors", "ark_m1_fp64_issue_rate", "ark_m1_apply_preconditioner", "ark_m1_apply_operator_pair", "ark_m1_device_bytes",
    "ark_m1_last_error", "ark_m1_version",
    "ark_m1_slab_range", "ark_m1_group_create_local", "ark_m1_group_create_host", "ark_m1_nccl_unique_id", "ark_m1_group_create_nccl",
    "ark_m1_group_destroy", "ark_m1_group_set_stream", "ark_m1_group_local_slabs", "ark_m1_group_slab", "ark_m1_group_step_explicit",
    "ark_m1_group_step_implicit", "ark_m1_group_comm_stats", "ark_m1_group_last_error",
    "ark_m1_3d_create", "ark_m1_3d_destroy", "ark_m1_3d_set_stream", "ark_m1_3d_set_state", "ark_m1_3d_set_option", "ark_m1_3d_get_state", "ark_m1_3d_step_explicit",
    "ark_m1_3d_step_implicit", "ark_m1_3d_apply_operator", "ark_m1_3d_kernel_launches", "ark_m1_3d_last_error",
    "ark_m1_noalloc_setup", "ark_m1_noalloc_max_cells", "ark_m1_count_unrealizable_noalloc", "ark_m1_noalloc_last_error",
]


class ArkBc(C.Structure):
    _fields_ = [("xlo", C.c_int), ("xhi", C.c_int), ("ylo", C.c_int), ("yhi", C.c_int)]


_SENDRECV = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double),
                        C.POINTER(C.c_double), C.c_longlong)
_ALLREDUCE = C.CFUNCTYPE(C.c_int, C.c_void_p, C.POINTER(C.c_double), C.c_int)


class ArkBc3(C.Structure):
    _fields_ = [("xlo", C.c_int), ("xhi", C.c_int), ("ylo", C.c_int), ("yhi", C.c_int), ("zlo", C.c_int), ("zhi", C.c_int)]


class ArkHostTransport(C.Structure):
    _fields_ = [("ctx", C.c_void_p), ("sendrecv", _SENDRECV), ("allreduce_sum", _ALLREDUCE)]


_lib = None


def load_library(path: str | None = None):
    """dlopen libark_m1.so and declare the prototypes.  Raises if the library is missing (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError(f"{path} not found: build it with `python -m paper_2011_13926_b200.build` "
                           "(the CUDA library is the only implementation; there is no CPU fallback)")
    L = C.CDLL(path)
    vp, dp, d, i = C.c_void_p, C.c_void_p, C.c_double, C.c_int   # array pointers are passed as raw addresses
    L.ark_m1_create.restype = vp
    L.ark_m1_create.argtypes = [i, i, d, d, d, C.POINTER(ArkBc)]
    L.ark_m1_destroy.restype = None
    L.ark_m1_destroy.argtypes = [vp]
    L.ark_m1_set_stream.argtypes = [vp, vp]
    L.ark_m1_set_state.argtypes = [vp, dp, dp, dp, dp, dp]
    L.ark_m1_set_boundary.argtypes = [vp, i, dp, dp, dp, dp]
    L.ark_m1_set_option.argtypes = [vp, C.c_char_p, d]
    L.ark_m1_set_field.argtypes = [vp, C.c_char_p, dp]
    L.ark_m1_get_state.argtypes = [vp, dp, dp, dp]
    L.ark_m1_prefetch_state.argtypes = [vp, dp, dp, dp, dp]
    L.ark_m1_commit_state.argtypes = [vp]
    L.ark_m1_get_state_async.argtypes = [vp, dp, dp]
    L.ark_m1_wait_transfers.argtypes = [vp]
    L.ark_m1_step_explicit.argtypes = [vp, d]
    L.ark_m1_steps_explicit.argtypes = [vp, d, i]
    L.ark_m1_step_implicit.argtypes = [vp, d, d, i, i, C.POINTER(C.c_double)]
    L.ark_m1_step_semi_implicit.argtypes = [vp, d, d, i, i, C.POINTER(C.c_double)]
    L.ark_m1_step_implicit_newton.argtypes = [vp, d, d, i, i, d, i, C.POINTER(C.c_int), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.ark_m1_add_velocity_sources.argtypes = [vp, d]
    L.ark_m1_count_unrealizable.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    L.ark_m1_residual.argtypes = [vp, dp, dp]
    L.ark_m1_apply_operator.argtypes = [vp, d, dp, dp, dp]
    L.ark_m1_apply_preconditioner.argtypes = [vp, d, dp, dp]
    L.ark_m1_apply_operator_pair.argtypes = [vp, d, dp, dp, dp, d, d]
    L.ark_m1_get_history.argtypes = [vp, C.POINTER(C.c_double), i]
    L.ark_m1_get_timings.argtypes = [vp, C.POINTER(C.c_double)]
    L.ark_m1_get_kernel_stats.argtypes = [vp, C.POINTER(C.c_double), i]
    L.ark_m1_kernel_class_name.restype = C.c_char_p
    L.ark_m1_kernel_class_name.argtypes = [i]
    L.ark_m1_kernel_launches.restype = C.c_longlong
    L.ark_m1_kernel_launches.argtypes = [vp]
    L.ark_m1_block_stats.restype = C.c_int
    L.ark_m1_block_stats.argtypes = [vp, C.POINTER(C.c_longlong)]
    L.ark_m1_fastmath_errors.argtypes = [i, C.POINTER(C.c_double)]
    L.ark_m1_fp64_issue_rate.argtypes = [C.POINTER(C.c_double), i]
    L.ark_m1_device_bytes.restype = C.c_longlong
    L.ark_m1_device_bytes.argtypes = [vp]
    L.ark_m1_last_error.restype = C.c_char_p
    L.ark_m1_last_error.argtypes = [vp]
    L.ark_m1_version.restype = C.c_char_p
    L.ark_m1_version.argtypes = []
    ip = C.POINTER(C.c_int)
    L.ark_m1_slab_range.argtypes = [i, i, i, ip, ip]
    L.ark_m1_group_create_local.restype = vp
    L.ark_m1_group_create_local.argtypes = [i, i, d, d, d, C.POINTER(ArkBc), i]
    L.ark_m1_group_create_host.restype = vp
    L.ark_m1_group_create_host.argtypes = [i, i, d, d, d, C.POINTER(ArkBc), i, i, C.POINTER(ArkHostTransport)]
    L.ark_m1_nccl_unique_id.argtypes = [vp]
    L.ark_m1_group_create_nccl.restype = vp
    L.ark_m1_group_create_nccl.argtypes = [i, i, d, d, d, C.POINTER(ArkBc), i, i, vp]
    L.ark_m1_group_destroy.restype = None
    L.ark_m1_group_destroy.argtypes = [vp]
    L.ark_m1_group_set_stream.argtypes = [vp, vp]
    L.ark_m1_group_local_slabs.argtypes = [vp]
    L.ark_m1_group_slab.restype = vp
    L.ark_m1_group_slab.argtypes = [vp, i, ip, ip, ip]
    L.ark_m1_group_step_explicit.argtypes = [vp, d]
    L.ark_m1_group_step_implicit.argtypes = [vp, d, d, i, i, C.POINTER(C.c_double)]
    L.ark_m1_group_comm_stats.argtypes = [vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    L.ark_m1_group_last_error.restype = C.c_char_p
    L.ark_m1_group_last_error.argtypes = [vp]
    L.ark_m1_3d_create.restype = vp
    L.ark_m1_3d_create.argtypes = [i, i, i, d, d, d, d, C.POINTER(ArkBc3)]
    L.ark_m1_3d_destroy.restype = None
    L.ark_m1_3d_destroy.argtypes = [vp]
    L.ark_m1_3d_set_stream.argtypes = [vp, vp]
    L.ark_m1_3d_set_state.argtypes = [vp, dp, dp, dp, dp]
    L.ark_m1_3d_set_option.argtypes = [vp, C.c_char_p, d]
    L.ark_m1_3d_get_state.argtypes = [vp, dp, dp]
    L.ark_m1_3d_step_explicit.argtypes = [vp, d]
    L.ark_m1_3d_step_implicit.argtypes = [vp, d, d, i, i, C.POINTER(C.c_double)]
    L.ark_m1_3d_apply_operator.argtypes = [vp, d, dp, dp, i]
    L.ark_m1_3d_kernel_launches.restype = C.c_longlong
    L.ark_m1_3d_kernel_launches.argtypes = [vp]
    L.ark_m1_3d_last_error.restype = C.c_char_p
    L.ark_m1_3d_last_error.argtypes = [vp]
    L.ark_m1_noalloc_setup.argtypes = []
    L.ark_m1_noalloc_max_cells.restype = C.c_longlong
    L.ark_m1_noalloc_max_cells.argtypes = []
    L.ark_m1_count_unrealizable_noalloc.argtypes = [dp, dp, dp, C.c_longlong, d, vp, vp]
    L.ark_m1_noalloc_last_error.restype = C.c_char_p
    L.ark_m1_noalloc_last_error.argtypes = []
    for name in SYMBOLS:
        getattr(L, name)
    _lib = L
    return L


def _ptr(a, nelem=None):
    """Raw address of a float64 contiguous torch tensor / numpy array (None -> NULL).  Returns (address, keepalive)."""
    if a is None:
        return None, None
    try:
        import torch
    except ImportError:  # numpy-only callers
        torch = None
    if torch is not None and isinstance(a, torch.Tensor):
        if a.dtype != torch.float64 or not a.is_contiguous():
            raise TypeError("tensor arguments must be contiguous float64")
        if nelem is not None and a.numel() != nelem:
            raise ValueError(f"expected {nelem} elements, got {a.numel()}")
        return a.data_ptr(), a
    arr = np.ascontiguousarray(a, dtype=np.float64)
    if nelem is not None and arr.size != nelem:
        raise ValueError(f"expected {nelem} elements, got {arr.size}")
    return arr.ctypes.data, arr


class ArkM1:
    """One solver handle.  Method names follow include/ark_m1.h without the ark_m1_ prefix."""

    def __init__(self, nx, ny, dx, dy, c=1.0, bc=(0, 0, 0, 0), stream=None, _borrowed=None):
        self._L = load_library()
        self.nx, self.ny, self.dx, self.dy, self.c = int(nx), int(ny), float(dx), float(dy), float(c)
        self.bc = tuple(int(b) for b in bc)
        self._owned = _borrowed is None
        if _borrowed is not None:          # a slab of an ArkM1Group: the group owns the handle
            self._h = _borrowed
            return
        b = ArkBc(*self.bc)
        self._h = self._L.ark_m1_create(self.nx, self.ny, self.dx, self.dy, self.c, C.byref(b))
        if not self._h:
            raise ValueError("ark_m1_create failed (bad arguments or no CUDA device)")
        if stream is not None:
            self.set_stream(stream)

    def close(self):
        if getattr(self, "_h", None):
            if self._owned:
                self._L.ark_m1_destroy(self._h)
            self._h = None

    __del__ = close

    def _check(self, rc):
        if rc < 0:
            raise RuntimeError(f"ark_m1 error {rc}: {self._L.ark_m1_last_error(self._h).decode()}")
        return rc

    @property
    def N(self):
        return self.nx * self.ny

    def set_stream(self, stream):
        """stream: a torch.cuda.Stream, or a raw cudaStream_t address."""
        addr = getattr(stream, "cuda_stream", stream)
        self._check(self._L.ark_m1_set_stream(self._h, C.c_void_p(addr)))

    def set_state(self, E, F, sigma_a, sigma_s, T=None):
        N = self.N
        pe, k0 = _ptr(E, N); pf, k1 = _ptr(F, 2 * N); pa, k2 = _ptr(sigma_a, N); ps, k3 = _ptr(sigma_s, N); pt, k4 = _ptr(T, N)
        self._check(self._L.ark_m1_set_state(self._h, pe, pf, pa, ps, pt))
        self._keep = (k0, k1, k2, k3, k4)   # sources of asynchronous copies stay alive until the next call

    def set_boundary(self, side, E_g, F_g, sigma_a_g, sigma_s_g):
        n = self.ny if side < 2 else self.nx
        pe, k0 = _ptr(E_g, n); pf, k1 = _ptr(F_g, 2 * n); pa, k2 = _ptr(sigma_a_g, n); ps, k3 = _ptr(sigma_s_g, n)
        self._check(self._L.ark_m1_set_boundary(self._h, int(side), pe, pf, pa, ps))
        self._keep_b = getattr(self, "_keep_b", []) + [(k0, k1, k2, k3)]

    def set_option(self, key, value):
        self._check(self._L.ark_m1_set_option(self._h, key.encode(), float(value)))

    def set_field(self, name, plane):
        p, k = _ptr(plane, self.N)
        self._check(self._L.ark_m1_set_field(self._h, name.encode(), p))
        self._keep_f = getattr(self, "_keep_f", []) + [k]

    def get_state(self, with_T=False, out=None):
        """Returns numpy arrays E[ny,nx], F[2,ny,nx] (and T) unless `out` = (E, F[, T]) buffers are given."""
        if out is None:
            E = np.empty((self.ny, self.nx)); F = np.empty((2, self.ny, self.nx))
            T = np.empty((self.ny, self.nx)) if with_T else None
        else:
            E, F = out[0], out[1]
            T = out[2] if len(out) > 2 else None
        pe, _ = _ptr(E, self.N); pf, _ = _ptr(F, 2 * self.N); pt, _ = _ptr(T, self.N)
        self._check(self._L.ark_m1_get_state(self._h, pe, pf, pt))
        return (E, F, T) if (with_T or (out is not None and len(out) > 2)) else (E, F)

    # ---- overlapped transfers (csrc/pipeline.cu): the next state goes up and the last result comes down beside the running solve
    def prefetch_state(self, E, F, sigma_a, sigma_s):
        """Starts the upload of the NEXT state into a staging buffer on the handle's copy stream; returns at once."""
        N = self.N
        pe, k0 = _ptr(E, N); pf, k1 = _ptr(F, 2 * N); pa, k2 = _ptr(sigma_a, N); ps, k3 = _ptr(sigma_s, N)
        self._check(self._L.ark_m1_prefetch_state(self._h, pe, pf, pa, ps))
        self._keep_up = (k0, k1, k2, k3)

    def commit_state(self):
        """The handle's stream waits for the prefetched upload and takes the staged state (radiation-only: T unset)."""
        self._check(self._L.ark_m1_commit_state(self._h))

    def get_state_async(self, out):
        """Snapshot of the current state copied to out = (E, F) on the copy stream; valid after wait_transfers()."""
        pe, k0 = _ptr(out[0], self.N); pf, k1 = _ptr(out[1], 2 * self.N)
        self._check(self._L.ark_m1_get_state_async(self._h, pe, pf))
        self._keep_down = (k0, k1)

    def wait_transfers(self):
        self._check(self._L.ark_m1_wait_transfers(self._h))

    def step_explicit(self, dt):
        self._check(self._L.ark_m1_step_explicit(self._h, float(dt)))

    def steps_explicit(self, dt, nsteps):
        self._check(self._L.ark_m1_steps_explicit(self._h, float(dt), int(nsteps)))

    def step_implicit(self, dt, tol=1e-10, restart=30, maxit=4000):
        res = C.c_double(0.0)
        its = self._check(self._L.ark_m1_step_implicit(self._h, float(dt), float(tol), int(restart), int(maxit), C.byref(res)))
        return its, res.value

    def step_semi_implicit(self, dt, tol=1e-12, restart=30, maxit=4000):
        res = C.c_double(0.0)
        its = self._check(self._L.ark_m1_step_semi_implicit(self._h, float(dt), float(tol), int(restart), int(maxit), C.byref(res)))
        return its, res.value

    def step_implicit_newton(self, dt, tol=1e-10, restart=30, maxit=4000, newton_tol=1e-8, max_newton=20):
        """Returns (total GMRES iterations, Newton iterations, last true relative residual, last relative update)."""
        nn, res, upd = C.c_int(0), C.c_double(0.0), C.c_double(0.0)
        its = self._check(self._L.ark_m1_step_implicit_newton(self._h, float(dt), float(tol), int(restart), int(maxit), float(newton_tol),
                                                              int(max_newton), C.byref(nn), C.byref(res), C.byref(upd)))
        return its, nn.value, res.value, upd.value

    def add_velocity_sources(self, dt):
        self._check(self._L.ark_m1_add_velocity_sources(self._h, float(dt)))

    def count_unrealizable(self):
        a, b = C.c_longlong(0), C.c_longlong(0)
        self._check(self._L.ark_m1_count_unrealizable(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def residual(self):
        RE = np.empty((self.ny, self.nx)); RF = np.empty((2, self.ny, self.nx))
        self._check(self._L.ark_m1_residual(self._h, RE.ctypes.data, RF.ctypes.data))
        return RE, RF

    def apply_operator(self, dt, V, with_b=False):
        p, keep = _ptr(V, 3 * self.N)
        out = np.empty((3, self.ny, self.nx))
        b = np.empty((3, self.ny, self.nx)) if with_b else None
        self._check(self._L.ark_m1_apply_operator(self._h, float(dt), p, out.ctypes.data, None if b is None else b.ctypes.data))
        return (out, b) if with_b else out

    def apply_preconditioner(self, dt, V):
        p, keep = _ptr(V, 3 * self.N)
        out = np.empty((3, self.ny, self.nx))
        self._check(self._L.ark_m1_apply_preconditioner(self._h, float(dt), p, out.ctypes.data))
        return out

    def apply_operator_pair(self, dt, V, theta1=0.0, theta2=0.0):
        """(out1, out2, fused): out1 = A M^-1 V - theta1 V, out2 = A M^-1 out1 - theta2 out1; fused = the one-pass kernel ran."""
        p, keep = _ptr(V, 3 * self.N)
        o1 = np.empty((3, self.ny, self.nx)); o2 = np.empty((3, self.ny, self.nx))
        fused = self._check(self._L.ark_m1_apply_operator_pair(self._h, float(dt), p, o1.ctypes.data, o2.ctypes.data, float(theta1), float(theta2)))
        return o1, o2, bool(fused)

    def history(self):
        n = self._L.ark_m1_get_history(self._h, None, 0)
        buf = (C.c_double * max(n, 1))()
        self._L.ark_m1_get_history(self._h, buf, n)
        return np.array(buf[:n])

    def timings(self):
        buf = (C.c_double * 3)()
        self._check(self._L.ark_m1_get_timings(self._h, buf))
        return dict(assembly_ms=buf[0], krylov_ms=buf[1], total_ms=buf[2])

    def kernel_stats(self):
        """{class name: dict(launches, ms, bytes)} since set_option("kernel_timing", 1)."""
        buf = (C.c_double * 64)()
        n = self._check(self._L.ark_m1_get_kernel_stats(self._h, buf, 64))
        return {self._L.ark_m1_kernel_class_name(k).decode(): dict(launches=int(buf[3 * k]), ms=buf[3 * k + 1], bytes=buf[3 * k + 2])
                for k in range(n)}

    def kernel_launches(self):
        return int(self._L.ark_m1_kernel_launches(self._h))

    def block_stats(self):
        """s-step Arnoldi blocks of the last linear solve: dict(update_pass, predicted_refined, separate_pass, separate_refined)."""
        buf = (C.c_longlong * 4)()
        self._check(self._L.ark_m1_block_stats(self._h, buf))
        return dict(update_pass=int(buf[0]), predicted_refined=int(buf[1]), separate_pass=int(buf[2]), separate_refined=int(buf[3]))

    def device_bytes(self):
        return int(self._L.ark_m1_device_bytes(self._h))


def slab_range(ny, nranks, rank):
    """Rows [y0, y1) of slab `rank` (ark_m1_slab_range; host arithmetic, works without a GPU)."""
    y0, y1 = C.c_int(0), C.c_int(0)
    if load_library().ark_m1_slab_range(int(ny), int(nranks), int(rank), C.byref(y0), C.byref(y1)) < 0:
        raise ValueError("ark_m1_slab_range: bad arguments")
    return y0.value, y1.value


def gloo_host_transport(dist, rank, nranks):
    """ArkHostTransport whose callbacks move the host buffers with torch.distributed (any backend with CPU tensors, e.g. gloo).
    Returns (transport struct, keepalive)."""
    import torch

    def _view(ptr, n):
        return torch.from_numpy(np.ctypeslib.as_array(ptr, shape=(int(n),)))

    def sendrecv(ctx, lo, hi, send_lo, send_hi, recv_lo, recv_hi, n):
        try:
            ops, keep = [], []
            # what goes to `lo` is that rank's upper halo (tag 1); what goes to `hi` is its lower halo (tag 0)
            if lo >= 0:
                t = _view(send_lo, n).clone(); keep.append(t); ops.append(dist.P2POp(dist.isend, t, lo, tag=1))
            if hi >= 0:
                t = _view(send_hi, n).clone(); keep.append(t); ops.append(dist.P2POp(dist.isend, t, hi, tag=0))
            rl = rh = None
            if hi >= 0:
                rh = torch.empty(int(n), dtype=torch.float64); ops.append(dist.P2POp(dist.irecv, rh, hi, tag=1))
            if lo >= 0:
                rl = torch.empty(int(n), dtype=torch.float64); ops.append(dist.P2POp(dist.irecv, rl, lo, tag=0))
            if ops:
                for req in dist.batch_isend_irecv(ops):
                    req.wait()
            if rl is not None:
                _view(recv_lo, n).copy_(rl)
            if rh is not None:
                _view(recv_hi, n).copy_(rh)
            return 0
        except Exception as exc:      # never let an exception cross the C boundary
            print(f"gloo_host_transport.sendrecv failed on rank {rank}: {exc!r}")
            return -1

    def allreduce(ctx, buf, n):
        try:
            t = _view(buf, n).clone()
            dist.all_reduce(t)
            _view(buf, n).copy_(t)
            return 0
        except Exception as exc:
            print(f"gloo_host_transport.allreduce failed on rank {rank}: {exc!r}")
            return -1

    cb1, cb2 = _SENDRECV(sendrecv), _ALLREDUCE(allreduce)
    return ArkHostTransport(None, cb1, cb2), (cb1, cb2)


class ArkM1Group:
    """Slab-decomposed solver (include/ark_m1.h, "Domain-decomposed step").  kind = "local" (all slabs in this process, one
    GPU), "host" (one slab per process, `transport` = ArkHostTransport) or "nccl" (one slab per process and GPU,
    `unique_id` = the 128 bytes of nccl_unique_id() of one rank)."""

    def __init__(self, nx, ny, dx, dy, c=1.0, bc=(0, 0, 0, 0), nranks=1, kind="local", rank=0, transport=None, unique_id=None, stream=None):
        self._L = load_library()
        self.nx, self.ny, self.nranks, self.rank, self.kind = int(nx), int(ny), int(nranks), int(rank), kind
        b = ArkBc(*[int(v) for v in bc])
        self._keep = transport
        if kind == "local":
            self._g = self._L.ark_m1_group_create_local(self.nx, self.ny, float(dx), float(dy), float(c), C.byref(b), self.nranks)
        elif kind == "host":
            self._g = self._L.ark_m1_group_create_host(self.nx, self.ny, float(dx), float(dy), float(c), C.byref(b), self.rank, self.nranks,
                                                       C.byref(transport[0] if isinstance(transport, tuple) else transport))
        elif kind == "nccl":
            self._idbuf = C.create_string_buffer(bytes(unique_id), 128)
            self._g = self._L.ark_m1_group_create_nccl(self.nx, self.ny, float(dx), float(dy), float(c), C.byref(b), self.rank, self.nranks,
                                                       C.cast(self._idbuf, C.c_void_p))
        else:
            raise ValueError("kind must be local, host or nccl")
        if not self._g:
            raise ValueError("ark_m1_group_create failed (bad arguments, no CUDA device, or the transport could not be set up)")
        self.slabs = []
        for k in range(self._L.ark_m1_group_local_slabs(self._g)):
            r, y0, y1 = C.c_int(0), C.c_int(0), C.c_int(0)
            h = self._L.ark_m1_group_slab(self._g, k, C.byref(r), C.byref(y0), C.byref(y1))
            s = ArkM1(self.nx, y1.value - y0.value, dx, dy, c, bc, _borrowed=h)
            s.rank, s.y0, s.y1 = r.value, y0.value, y1.value
            self.slabs.append(s)
        if stream is not None:
            self.set_stream(stream)

    def close(self):
        if getattr(self, "_g", None):
            for s in self.slabs:
                s.close()
            self._L.ark_m1_group_destroy(self._g)
            self._g = None

    __del__ = close

    def _check(self, rc):
        if rc < 0:
            raise RuntimeError(f"ark_m1_group error {rc}: {self._L.ark_m1_group_last_error(self._g).decode()}")
        return rc

    def set_stream(self, stream):
        addr = getattr(stream, "cuda_stream", stream)
        self._check(self._L.ark_m1_group_set_stream(self._g, C.c_void_p(addr)))

    def set_option(self, key, value):
        for s in self.slabs:
            s.set_option(key, value)

    def scatter(self, w):
        """Give every local slab its rows of a GLOBAL workload dict (E, F, sigma_a, sigma_s[, T, rho_cv, source_E, ux, uy], x-side
        ghosts per row, y-side ghosts on the end slabs)."""
        for s in self.slabs:
            rows = slice(s.y0, s.y1)
            cut = lambda a: None if a is None else np.ascontiguousarray(np.asarray(a)[..., rows, :])
            s.set_state(cut(w["E"]), cut(w["F"]), cut(w["sigma_a"]), cut(w["sigma_s"]), cut(w.get("T")))
            for name in ("rho_cv", "ux", "uy", "source_E"):
                if w.get(name) is not None:
                    s.set_field(name, cut(w[name]))
            for side, gh in (w.get("ghosts") or {}).items():
                if side < 2:           # x sides: one value per row of the slab
                    s.set_boundary(side, *[np.ascontiguousarray(np.asarray(a)[..., rows]) for a in gh])
                elif (side == 2 and s.y0 == 0) or (side == 3 and s.y1 == self.ny):
                    s.set_boundary(side, *gh)

    def gather(self, with_T=False):
        """Rows held by this process: list of (y0, y1, E, F[, T])."""
        return [(s.y0, s.y1) + tuple(s.get_state(with_T=with_T)) for s in self.slabs]

    def get_state(self, with_T=False):
        """The stitched global state (local groups only)."""
        parts = self.gather(with_T)
        E = np.concatenate([p[2] for p in parts], axis=0)
        F = np.concatenate([p[3] for p in parts], axis=1)
        return (E, F, np.concatenate([p[4] for p in parts], axis=0)) if with_T else (E, F)

    def step_explicit(self, dt):
        self._check(self._L.ark_m1_group_step_explicit(self._g, float(dt)))

    def step_implicit(self, dt, tol=1e-10, restart=30, maxit=4000):
        res = C.c_double(0.0)
        its = self._check(self._L.ark_m1_group_step_implicit(self._g, float(dt), float(tol), int(restart), int(maxit), C.byref(res)))
        return its, res.value

    def comm_stats(self):
        a, b, c_ = C.c_longlong(0), C.c_longlong(0), C.c_longlong(0)
        self._check(self._L.ark_m1_group_comm_stats(self._g, C.byref(a), C.byref(b), C.byref(c_)))
        return dict(halo_bytes=a.value, exchanges=b.value, allreduces=c_.value)


class ArkM1_3D:
    """The 3-D solver (include/ark_m1.h "Three space dimensions").  Arrays [nz, ny, nx]; F is [3, nz, ny, nx]."""

    def __init__(self, nx, ny, nz, dx, dy, dz, c=1.0, bc=(0, 0, 0, 0, 0, 0), stream=None):
        self._L = load_library()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        b = ArkBc3(*[int(v) for v in bc])
        self._h = self._L.ark_m1_3d_create(self.nx, self.ny, self.nz, float(dx), float(dy), float(dz), float(c), C.byref(b))
        if not self._h:
            raise ValueError("ark_m1_3d_create failed (bad arguments or no CUDA device)")
        if stream is not None:
            self._check(self._L.ark_m1_3d_set_stream(self._h, C.c_void_p(getattr(stream, "cuda_stream", stream))))

    def close(self):
        if getattr(self, "_h", None):
            self._L.ark_m1_3d_destroy(self._h)
            self._h = None

    __del__ = close

    def _check(self, rc):
        if rc < 0:
            raise RuntimeError(f"ark_m1_3d error {rc}: {self._L.ark_m1_3d_last_error(self._h).decode()}")
        return rc

    @property
    def N(self):
        return self.nx * self.ny * self.nz

    def set_state(self, E, F, sigma_a, sigma_s):
        N = self.N
        pe, k0 = _ptr(E, N); pf, k1 = _ptr(F, 3 * N); pa, k2 = _ptr(sigma_a, N); ps, k3 = _ptr(sigma_s, N)
        self._check(self._L.ark_m1_3d_set_state(self._h, pe, pf, pa, ps))
        self._keep = (k0, k1, k2, k3)

    def set_option(self, key, value):
        self._check(self._L.ark_m1_3d_set_option(self._h, key.encode(), float(value)))

    def get_state(self):
        E = np.empty((self.nz, self.ny, self.nx)); F = np.empty((3, self.nz, self.ny, self.nx))
        self._check(self._L.ark_m1_3d_get_state(self._h, E.ctypes.data, F.ctypes.data))
        return E, F

    def step_explicit(self, dt):
        self._check(self._L.ark_m1_3d_step_explicit(self._h, float(dt)))

    def step_implicit(self, dt, tol=1e-10, restart=30, maxit=4000):
        res = C.c_double(0.0)
        its = self._check(self._L.ark_m1_3d_step_implicit(self._h, float(dt), float(tol), int(restart), int(maxit), C.byref(res)))
        return its, res.value

    def apply_operator(self, dt, V, precond=False):
        p, keep = _ptr(V, 4 * self.N)
        out = np.empty((4, self.nz, self.ny, self.nx))
        self._check(self._L.ark_m1_3d_apply_operator(self._h, float(dt), p, out.ctypes.data, int(bool(precond))))
        return out

    def kernel_launches(self):
        return int(self._L.ark_m1_3d_kernel_launches(self._h))


def nccl_unique_id():
    buf = C.create_string_buffer(128)
    rc = load_library().ark_m1_nccl_unique_id(C.cast(buf, C.c_void_p))
    if rc < 0:
        raise RuntimeError(f"ark_m1_nccl_unique_id failed ({rc}): libnccl.so.2 not loadable?")
    return bytes(buf.raw)


def fastmath_errors(n=1 << 20):
    """Max relative errors (rcp_fast, rsqrt_fast, sqrt_fast, rcp_fast3) of the kernels' fast fp64 forms against IEEE, measured on the GPU."""
    buf = (C.c_double * 4)()
    rc = load_library().ark_m1_fastmath_errors(int(n), buf)
    if rc < 0:
        raise RuntimeError(f"ark_m1_fastmath_errors failed ({rc})")
    return tuple(buf)


PIPE_RATE_KEYS = ("dfma_lanes_per_clk_sm", "dfma_latency_cycles", "dadd_lanes_per_clk_sm", "dmul_lanes_per_clk_sm",
                  "dmax_sel_lanes_per_clk_sm", "imad_lanes_per_clk_sm", "ffma_lanes_per_clk_sm", "dfma_imad_pair_issue_cycles",
                  "dfma_ffma_pair_issue_cycles", "shfl64_lanes_per_clk_sm", "sm_mhz", "sm_count")


def fp64_issue_rate():
    """Issue rates measured on the current GPU by ark_m1_fp64_issue_rate (see include/ark_m1.h), as a dict."""
    buf = (C.c_double * 12)()
    rc = load_library().ark_m1_fp64_issue_rate(buf, 12)
    if rc < 0:
        raise RuntimeError(f"ark_m1_fp64_issue_rate failed ({rc})")
    return dict(zip(PIPE_RATE_KEYS, (float(v) for v in buf)))


def noalloc_setup():
    """Resolve the static scratch array of the no-allocation entry point on the current device (once per device, before a capture)."""
    L = load_library()
    rc = L.ark_m1_noalloc_setup()
    if rc < 0:
        raise RuntimeError(f"ark_m1_noalloc_setup failed ({rc}): {L.ark_m1_noalloc_last_error().decode()}")


def noalloc_max_cells():
    return int(load_library().ark_m1_noalloc_max_cells())


def count_unrealizable_noalloc(E, Fx, Fy, c, counts2, stream=None):
    """ark_m1_count_unrealizable_noalloc: E, Fx, Fy float64 CUDA tensors of equal size, counts2 a CUDA tensor of 2 x int64 (the two
    unsigned 64-bit counts), all on the current device.  Enqueues on `stream` (torch stream or raw address; default: torch's current
    stream) and returns without synchronising; allocates nothing."""
    import torch
    L = load_library()
    for t in (E, Fx, Fy):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == E.numel()):
            raise TypeError("E, Fx, Fy must be contiguous float64 CUDA tensors of equal size")
    if not (isinstance(counts2, torch.Tensor) and counts2.is_cuda and counts2.dtype == torch.int64 and counts2.is_contiguous() and counts2.numel() == 2):
        raise TypeError("counts2 must be a contiguous int64 CUDA tensor of 2 elements")
    st = torch.cuda.current_stream() if stream is None else stream
    st = getattr(st, "cuda_stream", st)
    n = E.numel()
    rc = L.ark_m1_count_unrealizable_noalloc(E.data_ptr() if n else None, Fx.data_ptr() if n else None, Fy.data_ptr() if n else None,
                                             n, float(c), counts2.data_ptr(), st)
    if rc < 0:
        raise RuntimeError(f"ark_m1 error {rc}: {L.ark_m1_noalloc_last_error().decode()}")


def version():
    return load_library().ark_m1_version().decode()
