"""Thin ctypes binding of libtpt.so (include/tpt.h).  Argument marshalling only — every step of the
solve runs in the library's CUDA kernels.  PyTorch is used for device memory and streams.

    plan = plan_create(nx, ny, nz, xf, yf, zf, bc, helmholtz_alpha)
    solve(plan, rhs, out)            # torch.float64 CUDA tensors of nx*ny*nz elements
    plan_destroy(plan)

Fails loudly (RuntimeError) if the library has not been built or a call returns a non-zero status.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libtpt.so")

NEUMANN, DIRICHLET, PERIODIC = 0, 1, 2
DIRS_Z, DIRS_YZ, DIRS_XYZ = 4, 6, 7   # implicitly treated directions of Eq. 2b: bit 0 = x, 1 = y, 2 = z
K_FWD_X, K_FWD_Y, K_THOMAS, K_INV_Y, K_INV_X, K_COUNT = 0, 1, 2, 3, 4, 5
KERNEL_NAMES = ("fwd_x", "fwd_y", "thomas", "inv_y", "inv_x")
# tpt_plan_get_paths codes
(PATH_NONE, PATH_GEMM_GENERIC, PATH_GEMM_CPASYNC, PATH_GEMM_TMA, PATH_FFT, PATH_THOMAS_STREAM, PATH_THOMAS_ONCHIP,
 PATH_THOMAS_BLOCKED, PATH_FUSED_SMALL) = range(9)

# every symbol include/tpt.h declares (tests check the library exports exactly these)
TRANSFORM_GEMM, TRANSFORM_FFT = 0, 1   # per diagonalised direction: eigenbasis GEMM / fast transform

SYMBOLS = (
    "tpt_plan_create", "tpt_plan_create_dirs", "tpt_solve", "tpt_solve_static_scratch", "tpt_solve_batch", "tpt_plan_reserve_batch", "tpt_solve_host", "tpt_plan_destroy", "tpt_plan_get_eigen",
    "tpt_plan_is_singular", "tpt_plan_device_bytes", "tpt_stage", "tpt_plan_set_profiling",
    "tpt_plan_get_kernel_times", "tpt_plan_get_paths", "tpt_plan_launches", "tpt_plan_set_slab_groups", "tpt_plan_set_fused_small", "tpt_plan_set_gemm_variant", "tpt_plan_set_thomas_variant", "tpt_fp64_peak", "tpt_strerror", "tpt_version",
    "tpt_divergence", "tpt_gradient_correct", "tpt_project", "tpt_plan_create_ex", "tpt_solve_host_async", "tpt_plan_wait",
    "tpt_host_eigen", "tpt_debug_set_eigen_base", "tpt_debug_sweep_geometry", "tpt_fill_uniform",
    "tpt_shard_layout", "tpt_shard_create", "tpt_shard_create_ex", "tpt_shard_get_layout", "tpt_shard_sym", "tpt_shard_set_peers", "tpt_shard_ipc_export",
    "tpt_shard_ipc_import", "tpt_solve_sharded", "tpt_shard_solve_phase", "tpt_shard_barrier", "tpt_shard_barrier_all", "tpt_shard_launches", "tpt_shard_destroy",
)
IPC_HANDLE_BYTES = 64
STATIC_SCRATCH_POINTS = 16384   # TPT_STATIC_SCRATCH_POINTS
ELIMIT = -5                     # TPT_ELIMIT


class ShardLayout(C.Structure):
    """tpt_shard_layout_t of include/tpt.h."""
    _fields_ = [("rank", C.c_int), ("nranks", C.c_int), ("k0", C.c_int), ("k1", C.c_int), ("m0", C.c_int), ("m1", C.c_int),
                ("mode_bytes", C.c_size_t), ("slab_bytes", C.c_size_t), ("sym_bytes", C.c_size_t), ("slab_points", C.c_size_t),
                ("nvlink_bytes_per_solve", C.c_size_t)]


_dp = C.POINTER(C.c_double)
_lib = None


class TptError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: status {status} ({strerror(status)})")


def lib():
    """Load libtpt.so.  No fallback: a missing library is an error."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2603_09528_b200.build` "
                "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i, d = C.c_void_p, C.c_int, C.c_double
        L.tpt_plan_create.argtypes = [C.POINTER(vp), i, i, i, _dp, _dp, _dp, C.POINTER(i), d]
        L.tpt_plan_create_dirs.argtypes = [C.POINTER(vp), i, i, i, _dp, _dp, _dp, C.POINTER(i), d, i]
        L.tpt_plan_create_ex.argtypes = [C.POINTER(vp), i, i, i, _dp, _dp, _dp, C.POINTER(i), d, i, C.POINTER(i)]
        L.tpt_solve.argtypes = [vp, vp, vp, vp]
        L.tpt_solve_static_scratch.argtypes = [vp, vp, vp, vp]
        L.tpt_solve_batch.argtypes = [vp, vp, vp, i, vp]
        L.tpt_plan_reserve_batch.argtypes = [vp, i]
        L.tpt_solve_host.argtypes = [vp, vp, vp, vp]
        L.tpt_solve_host_async.argtypes = [vp, vp, vp, vp]
        L.tpt_plan_wait.argtypes = [vp]
        L.tpt_divergence.argtypes = [vp, vp, vp, vp, d, vp, vp]
        L.tpt_gradient_correct.argtypes = [vp, vp, d, vp, vp, vp, vp, d, i, vp]
        L.tpt_project.argtypes = [vp, vp, vp, vp, d, vp, vp, d, i, vp]
        L.tpt_plan_destroy.argtypes = [vp]
        L.tpt_plan_get_eigen.argtypes = [vp, i, _dp, _dp]
        L.tpt_plan_is_singular.argtypes = [vp]
        L.tpt_host_eigen.argtypes = [i, _dp, i, i, _dp, _dp]
        L.tpt_debug_set_eigen_base.argtypes = [i]
        L.tpt_debug_sweep_geometry.argtypes = [i, i, i, C.POINTER(i)]
        L.tpt_plan_device_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
        L.tpt_stage.argtypes = [vp, i, vp, vp, vp]
        L.tpt_plan_set_profiling.argtypes = [vp, i]
        L.tpt_plan_get_kernel_times.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(i), C.POINTER(i)]
        L.tpt_plan_get_paths.argtypes = [vp, C.POINTER(C.c_int)]
        L.tpt_plan_set_gemm_variant.argtypes = [vp, i]
        L.tpt_plan_set_fused_small.argtypes = [vp, i]
        L.tpt_plan_launches.argtypes = [vp]
        L.tpt_plan_set_slab_groups.argtypes = [vp, i]
        L.tpt_plan_set_thomas_variant.argtypes = [vp, i]
        L.tpt_fp64_peak.argtypes = [i, _dp]
        L.tpt_fill_uniform.argtypes = [vp, C.c_size_t, C.c_ulonglong, C.c_ulonglong, vp]
        L.tpt_shard_layout.argtypes = [i, i, i, i, i, C.POINTER(ShardLayout)]
        L.tpt_shard_create.argtypes = [C.POINTER(vp), i, i, i, i, i, _dp, _dp, _dp, C.POINTER(i), d, i]
        L.tpt_shard_create_ex.argtypes = [C.POINTER(vp), i, i, i, i, i, _dp, _dp, _dp, C.POINTER(i), d, C.POINTER(i)]
        L.tpt_shard_get_layout.argtypes = [vp, C.POINTER(ShardLayout)]
        L.tpt_shard_sym.argtypes = [vp, C.POINTER(vp), C.POINTER(C.c_size_t)]
        L.tpt_shard_set_peers.argtypes = [vp, C.POINTER(vp)]
        L.tpt_shard_ipc_export.argtypes = [vp, vp]
        L.tpt_shard_ipc_import.argtypes = [vp, vp]
        L.tpt_solve_sharded.argtypes = [vp, vp, vp, vp]
        L.tpt_shard_solve_phase.argtypes = [vp, i, vp, vp, vp]
        L.tpt_shard_barrier.argtypes = [vp, vp]
        L.tpt_shard_barrier_all.argtypes = [C.POINTER(vp), i, vp]
        L.tpt_shard_launches.argtypes = [vp]
        L.tpt_shard_destroy.argtypes = [vp]
        L.tpt_strerror.argtypes = [i]
        L.tpt_strerror.restype = C.c_char_p
        L.tpt_version.argtypes = []
        L.tpt_version.restype = C.c_char_p
        _lib = L
    return _lib


def strerror(status: int) -> str:
    return lib().tpt_strerror(int(status)).decode()


def version() -> str:
    return lib().tpt_version().decode()


def _check(status: int, what: str):
    if status != 0:
        raise TptError(status, what)


def _faces(x):
    a = np.ascontiguousarray(x, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _stream_handle(stream) -> C.c_void_p:
    if stream is None:
        import torch

        stream = torch.cuda.current_stream()
    return C.c_void_p(int(getattr(stream, "cuda_stream", stream)))


def _dev_ptr(t, count: int, what: str) -> C.c_void_p:
    import torch

    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
            and t.numel() == count):
        raise ValueError(f"{what}: need a contiguous CUDA float64 tensor of {count} elements")
    return C.c_void_p(t.data_ptr())


class Plan:
    """Handle of a tpt_plan.  Fields are float64 CUDA tensors of shape (nz, ny, nx) (x contiguous)."""

    def __init__(self, handle, nx, ny, nz):
        self._h = handle
        self.nx, self.ny, self.nz = nx, ny, nz

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def points(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def singular(self) -> bool:
        r = lib().tpt_plan_is_singular(self._h)
        if r < 0:
            raise TptError(r, "tpt_plan_is_singular")
        return bool(r)

    def eigen(self, direction: int):
        n = self.nx if direction == 0 else self.ny
        lam, q = np.empty(n), np.empty((n, n))
        _check(lib().tpt_plan_get_eigen(self._h, direction, lam.ctypes.data_as(_dp), q.ctypes.data_as(_dp)),
               "tpt_plan_get_eigen")
        return lam, q

    def eigenvalues(self, direction: int):
        """lambda only (also available for a fast-transform direction, whose basis is not stored)."""
        lam = np.empty(self.nx if direction == 0 else self.ny)
        _check(lib().tpt_plan_get_eigen(self._h, direction, lam.ctypes.data_as(_dp), None), "tpt_plan_get_eigen")
        return lam

    def device_bytes(self) -> int:
        b = C.c_size_t()
        _check(lib().tpt_plan_device_bytes(self._h, C.byref(b)), "tpt_plan_device_bytes")
        return int(b.value)

    def solve(self, rhs, out, stream=None):
        return solve(self, rhs, out, stream)

    def solve_static_scratch(self, rhs, out, stream=None):
        """tpt_solve_static_scratch: the one-launch solve with its scratch in a static device array (no allocation);
        grids of at most STATIC_SCRATCH_POINTS points."""
        _check(lib().tpt_solve_static_scratch(self._h, _dev_ptr(rhs, self.points, "rhs"), _dev_ptr(out, self.points, "out"),
                                              _stream_handle(stream)), "tpt_solve_static_scratch")
        return out

    def solve_host(self, rhs_host, out_host, stream=None):
        return solve_host(self, rhs_host, out_host, stream)

    def solve_batch(self, rhs, out, stream=None):
        return solve_batch(self, rhs, out, stream)

    def reserve_batch(self, nrhs: int):
        _check(lib().tpt_plan_reserve_batch(self._h, int(nrhs)), "tpt_plan_reserve_batch")

    def stage(self, slot: int, inp, out, stream=None):
        _check(lib().tpt_stage(self._h, slot, _dev_ptr(inp, self.points, "in"), _dev_ptr(out, self.points, "out"),
                               _stream_handle(stream)), "tpt_stage")
        return out

    def set_profiling(self, enabled: bool):
        _check(lib().tpt_plan_set_profiling(self._h, int(bool(enabled))), "tpt_plan_set_profiling")

    def kernel_times(self):
        """(mean ms per kernel slot [5], total launches, solves) over the profiled solves since the last
        read-out; synchronises on the last of them and resets the accumulation."""
        ms = (C.c_float * K_COUNT)()
        n, k = C.c_int(), C.c_int()
        _check(lib().tpt_plan_get_kernel_times(self._h, ms, C.byref(n), C.byref(k)), "tpt_plan_get_kernel_times")
        return [float(v) for v in ms], int(n.value), int(k.value)

    def paths(self):
        """The kernel each slot of a solve runs (PATH_* codes), with the plan's current variant settings."""
        out = (C.c_int * K_COUNT)()
        _check(lib().tpt_plan_get_paths(self._h, out), "tpt_plan_get_paths")
        return [int(v) for v in out]

    def launches_last(self) -> int:
        """Kernel launches enqueued by the last solve on this plan."""
        n = lib().tpt_plan_launches(self._h)
        if n < 0:
            raise TptError(n, "tpt_plan_launches")
        return int(n)

    def set_slab_groups(self, groups: int):
        """-1 automatic, 0 off, G > 0: run steps 2.2-2.4 through L2-resident slabs of G 16-column groups."""
        _check(lib().tpt_plan_set_slab_groups(self._h, int(groups)), "tpt_plan_set_slab_groups")

    def set_fused_small(self, enabled: bool):
        _check(lib().tpt_plan_set_fused_small(self._h, int(bool(enabled))), "tpt_plan_set_fused_small")

    def set_gemm_variant(self, variant: int):
        _check(lib().tpt_plan_set_gemm_variant(self._h, int(variant)), "tpt_plan_set_gemm_variant")

    def set_thomas_variant(self, variant: int):
        _check(lib().tpt_plan_set_thomas_variant(self._h, int(variant)), "tpt_plan_set_thomas_variant")

    def destroy(self):
        if self._h is not None:
            h, self._h = self._h, None
            _check(lib().tpt_plan_destroy(h), "tpt_plan_destroy")

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def plan_create(nx, ny, nz, xf, yf, zf, bc, helmholtz_alpha: float = 0.0, dirs: int = DIRS_XYZ,
                transform=(TRANSFORM_GEMM, TRANSFORM_GEMM)) -> Plan:
    xa, xp = _faces(xf)
    ya, yp = _faces(yf)
    za, zp = _faces(zf)
    if (xa.size, ya.size, za.size) != (nx + 1, ny + 1, nz + 1):
        raise ValueError("face arrays must have n+1 entries per direction")
    bca = (C.c_int * 3)(*[int(b) for b in bc])
    h = C.c_void_p()
    tra = (C.c_int * 2)(*[int(t) for t in transform])
    _check(lib().tpt_plan_create_ex(C.byref(h), nx, ny, nz, xp, yp, zp, bca, float(helmholtz_alpha), int(dirs), tra),
           "tpt_plan_create_ex")
    return Plan(h, nx, ny, nz)


def solve(plan: Plan, rhs, out, stream=None):
    """Enqueue one solve on `stream` (default: torch's current stream).  Asynchronous."""
    _check(lib().tpt_solve(plan._h, _dev_ptr(rhs, plan.points, "rhs"), _dev_ptr(out, plan.points, "out"),
                           _stream_handle(stream)), "tpt_solve")
    return out


def solve_batch(plan: Plan, rhs, out, stream=None):
    """Enqueue nrhs solves of stacked fields: rhs / out are CUDA float64 tensors of nrhs * nx*ny*nz elements."""
    nrhs, rem = divmod(rhs.numel(), plan.points)
    if rem or nrhs < 1:
        raise ValueError("rhs must hold a whole number of fields")
    _check(lib().tpt_solve_batch(plan._h, _dev_ptr(rhs, nrhs * plan.points, "rhs"), _dev_ptr(out, nrhs * plan.points, "out"),
                                 nrhs, _stream_handle(stream)), "tpt_solve_batch")
    return out


def solve_host(plan: Plan, rhs_host, out_host, stream=None, nowait: bool = False):
    """Solve with HOST buffers (numpy float64 arrays or CPU torch tensors, ideally pinned).  nowait: only enqueue
    (pinned buffers, kept valid until plan_wait); two plans on two streams then overlap their copies."""
    def hp(a, what):
        if isinstance(a, np.ndarray):
            if a.dtype != np.float64 or not a.flags["C_CONTIGUOUS"] or a.size != plan.points:
                raise ValueError(f"{what}: need a contiguous float64 array of {plan.points} elements")
            return C.c_void_p(a.ctypes.data)
        import torch

        if not (isinstance(a, torch.Tensor) and not a.is_cuda and a.dtype == torch.float64 and a.is_contiguous()
                and a.numel() == plan.points):
            raise ValueError(f"{what}: need a contiguous CPU float64 tensor of {plan.points} elements")
        return C.c_void_p(a.data_ptr())

    fn = lib().tpt_solve_host_async if nowait else lib().tpt_solve_host
    _check(fn(plan._h, hp(rhs_host, "rhs"), hp(out_host, "out"), _stream_handle(stream)), "tpt_solve_host")
    return out_host


def plan_wait(plan: Plan):
    """Block until the plan's most recent solve_host(..., nowait=True) has delivered its result."""
    _check(lib().tpt_plan_wait(plan._h), "tpt_plan_wait")


def face_counts(plan: Plan):
    """Element counts of the staggered velocity arrays u (nz, ny, nx+1), v (nz, ny+1, nx), w (nz+1, ny, nx)."""
    return ((plan.nx + 1) * plan.ny * plan.nz, plan.nx * (plan.ny + 1) * plan.nz, plan.nx * plan.ny * (plan.nz + 1))


def divergence(plan: Plan, u, v, w, out, scale: float = 1.0, stream=None):
    """out = scale * D(u, v, w) on the staggered grid (right-hand side of Eq. 2c).  Asynchronous."""
    cu, cv, cw = face_counts(plan)
    _check(lib().tpt_divergence(plan._h, _dev_ptr(u, cu, "u"), _dev_ptr(v, cv, "v"), _dev_ptr(w, cw, "w"), float(scale),
                                _dev_ptr(out, plan.points, "out"), _stream_handle(stream)), "tpt_divergence")
    return out


def gradient_correct(plan: Plan, phi, c: float, u, v, w, p=None, alpha_p: float = 0.0, dirs: int = DIRS_XYZ, stream=None):
    """u -= c G phi (Eq. 2d) and, if p is given, p += phi - alpha_p L_I phi (Eq. 2e).  In place, asynchronous."""
    cu, cv, cw = face_counts(plan)
    _check(lib().tpt_gradient_correct(plan._h, _dev_ptr(phi, plan.points, "phi"), float(c), _dev_ptr(u, cu, "u"),
                                      _dev_ptr(v, cv, "v"), _dev_ptr(w, cw, "w"),
                                      None if p is None else _dev_ptr(p, plan.points, "p"), float(alpha_p), int(dirs),
                                      _stream_handle(stream)), "tpt_gradient_correct")


def project(plan: Plan, u, v, w, gamma_dt: float, phi, p=None, alpha_p: float = 0.0, dirs: int = DIRS_XYZ, stream=None):
    """One pressure projection (Eq. 2c-2e) with a Poisson plan: u, v, w (and p) updated in place, phi = Phi."""
    cu, cv, cw = face_counts(plan)
    _check(lib().tpt_project(plan._h, _dev_ptr(u, cu, "u"), _dev_ptr(v, cv, "v"), _dev_ptr(w, cw, "w"), float(gamma_dt),
                             _dev_ptr(phi, plan.points, "phi"), None if p is None else _dev_ptr(p, plan.points, "p"),
                             float(alpha_p), int(dirs), _stream_handle(stream)), "tpt_project")
    return phi


def plan_destroy(plan: Plan):
    plan.destroy()


# ---- sharded solve (include/tpt.h "the solve sharded across the GPUs of one NVLink domain") ----------

def shard_layout(nranks: int, rank: int, nx: int, ny: int, nz: int) -> ShardLayout:
    """The z-slab / y-mode split of rank `rank` (host only, needs no device)."""
    lay = ShardLayout()
    _check(lib().tpt_shard_layout(int(nranks), int(rank), nx, ny, nz, C.byref(lay)), "tpt_shard_layout")
    return lay


class Shard:
    """Handle of a tpt_shard: rank `rank` of a solve sharded over `nranks` GPUs.  rhs / out are this rank's z-slab,
    float64 CUDA tensors of nx*ny*(k1-k0) elements, shape (k1-k0, ny, nx)."""

    def __init__(self, handle, nx, ny, nz):
        self._h = handle
        self.nx, self.ny, self.nz = nx, ny, nz
        lay = ShardLayout()
        _check(lib().tpt_shard_get_layout(handle, C.byref(lay)), "tpt_shard_get_layout")
        self.layout = lay

    @property
    def slab_shape(self):
        return (self.layout.k1 - self.layout.k0, self.ny, self.nx)

    @property
    def slab_points(self) -> int:
        return int(self.layout.slab_points)

    def sym(self):
        """(device pointer, bytes) of the symmetric allocation."""
        ptr, n = C.c_void_p(), C.c_size_t()
        _check(lib().tpt_shard_sym(self._h, C.byref(ptr), C.byref(n)), "tpt_shard_sym")
        return int(ptr.value), int(n.value)

    def set_peers(self, sym_ptrs):
        arr = (C.c_void_p * len(sym_ptrs))(*[C.c_void_p(int(q)) for q in sym_ptrs])
        _check(lib().tpt_shard_set_peers(self._h, arr), "tpt_shard_set_peers")

    def ipc_export(self) -> bytes:
        buf = C.create_string_buffer(IPC_HANDLE_BYTES)
        _check(lib().tpt_shard_ipc_export(self._h, buf), "tpt_shard_ipc_export")
        return buf.raw

    def ipc_import(self, handles):
        """handles: the nranks exported handles in rank order (bytes each)."""
        blob = b"".join(bytes(h) for h in handles)
        if len(blob) != IPC_HANDLE_BYTES * self.layout.nranks:
            raise ValueError("need one IPC handle per rank")
        _check(lib().tpt_shard_ipc_import(self._h, C.c_char_p(blob)), "tpt_shard_ipc_import")

    def _slab(self, t, what):
        return None if t is None else _dev_ptr(t, self.slab_points, what)

    def solve(self, rhs, out, stream=None):
        """The whole sharded solve of this rank's slab; every rank must call it (device-side barriers)."""
        _check(lib().tpt_solve_sharded(self._h, self._slab(rhs, "rhs"), self._slab(out, "out"), _stream_handle(stream)),
               "tpt_solve_sharded")
        return out

    def solve_phase(self, phase: int, rhs=None, out=None, stream=None):
        """One phase (0 forward + exchange 1, 1 sweep + exchange 2, 2 inverse) without any waiting kernel."""
        _check(lib().tpt_shard_solve_phase(self._h, int(phase), self._slab(rhs, "rhs"), self._slab(out, "out"),
                                           _stream_handle(stream)), "tpt_shard_solve_phase")

    def barrier(self, stream=None):
        _check(lib().tpt_shard_barrier(self._h, _stream_handle(stream)), "tpt_shard_barrier")

    def launches(self) -> int:
        return int(lib().tpt_shard_launches(self._h))

    def destroy(self):
        if self._h is not None:
            h, self._h = self._h, None
            _check(lib().tpt_shard_destroy(h), "tpt_shard_destroy")

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def shard_create(rank: int, nranks: int, nx, ny, nz, xf, yf, zf, bc, helmholtz_alpha: float = 0.0,
                 transform_x: int = TRANSFORM_GEMM, transform_y: int = TRANSFORM_GEMM) -> Shard:
    xa, xp = _faces(xf)
    ya, yp = _faces(yf)
    za, zp = _faces(zf)
    if (xa.size, ya.size, za.size) != (nx + 1, ny + 1, nz + 1):
        raise ValueError("face arrays must have n+1 entries per direction")
    bca = (C.c_int * 3)(*[int(b) for b in bc])
    h = C.c_void_p()
    tra = (C.c_int * 2)(int(transform_x), int(transform_y))
    _check(lib().tpt_shard_create_ex(C.byref(h), int(rank), int(nranks), nx, ny, nz, xp, yp, zp, bca, float(helmholtz_alpha),
                                     tra), "tpt_shard_create_ex")
    return Shard(h, nx, ny, nz)


def shard_barrier_all(shards, stream=None):
    """The flag barrier of all virtual ranks of one device as one cooperative launch (tpt_shard_barrier_all)."""
    arr = (C.c_void_p * len(shards))(*[s._h for s in shards])
    _check(lib().tpt_shard_barrier_all(arr, len(shards), _stream_handle(stream)), "tpt_shard_barrier_all")


def virtual_ranks_solve(shards, rhs_slabs, out_slabs, stream=None, barriers: bool = False):
    """Sharded solve with all ranks living on ONE device (virtual ranks): phase p of every rank, then phase p+1, on one
    stream — stream order stands in for the two flag barriers (barriers=True runs them as well, all ranks in one
    cooperative launch).  Pure call ordering; no arithmetic."""
    for ph in range(3):
        for s, r, o in zip(shards, rhs_slabs, out_slabs):
            s.solve_phase(ph, r if ph == 0 else None, o if ph == 2 else None, stream)
        if barriers and ph < 2:
            shard_barrier_all(shards, stream)
    return out_slabs


def host_eigen(faces, bc: int, base_kind: int = 0):
    """(lambda[n], qtilde[n, n]) from the plan-time eigen-solver alone (host only, no device needed)."""
    fa, fp = _faces(faces)
    n = fa.size - 1
    lam, q = np.empty(n), np.empty((n, n))
    _check(lib().tpt_host_eigen(n, fp, int(bc), int(base_kind), lam.ctypes.data_as(_dp), q.ctypes.data_as(_dp)), "tpt_host_eigen")
    return lam, q


SWEEP_GEOMETRY_KEYS = ("M", "cols", "max_threads", "ctas_per_sm", "table_in_smem", "S", "nbox", "box_rows", "buf_rows", "nbuf",
                       "threads", "smem")


def debug_sweep_geometry(nz: int, blocked: bool, sharded: bool = False):
    """tpt_debug_sweep_geometry as a dict (SWEEP_GEOMETRY_KEYS), or None where the on-chip sweep has no shape.  Host only."""
    out = (C.c_int * 12)()
    if lib().tpt_debug_sweep_geometry(int(nz), int(bool(blocked)), int(bool(sharded)), out) != 0:
        return None
    return dict(zip(SWEEP_GEOMETRY_KEYS, [int(v) for v in out]))


def debug_set_eigen_base(base_kind: int):
    """Base eigen-solver of plans created from now on: 0 = default, 1 = deliberately crude (tests only)."""
    _check(lib().tpt_debug_set_eigen_base(int(base_kind)), "tpt_debug_set_eigen_base")


def fill_uniform(out, seed: int, offset: int = 0, stream=None):
    """out[t] = seeded uniform[-1,1) white noise, bit-identical to inputs.uniform_pm1(seed, n, offset)."""
    _check(lib().tpt_fill_uniform(_dev_ptr(out, out.numel(), "out"), out.numel(), int(seed), int(offset),
                                  _stream_handle(stream)), "tpt_fill_uniform")
    return out


def fp64_peak(kind: int) -> float:
    """Measured FP64 pipe throughput in TFLOP/s: kind 0 = DFMA loop, 1 = DMMA loop."""
    v = C.c_double()
    _check(lib().tpt_fp64_peak(int(kind), C.byref(v)), "tpt_fp64_peak")
    return float(v.value)
