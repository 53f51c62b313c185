"""ctypes marshalling for oracle/libtpt_oracle.so (TEST INFRASTRUCTURE; no arithmetic here)."""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

DIRS_Z, DIRS_YZ, DIRS_XYZ = 4, 6, 7   # implicitly treated directions: bit 0 = x, 1 = y, 2 = z

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _ptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _bc(bc):
    return (C.c_int * 3)(*[int(b) for b in bc])


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_operator_1d.argtypes = [C.c_int, _dp, C.c_int, _dp, _dp, _dp, _dp]
        L.orc_symmetrize_1d.argtypes = [C.c_int, _dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_eig_1d.argtypes = [C.c_int, _dp, C.c_int, C.c_int, _dp, _dp]
        L.orc_plan_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, C.c_double]
        L.orc_plan_create_with_eig.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip,
                                               C.c_double, _dp, _dp, _dp, _dp]
        L.orc_plan_destroy.argtypes = [C.c_void_p]
        L.orc_plan_destroy.restype = None
        L.orc_plan_is_singular.argtypes = [C.c_void_p]
        L.orc_plan_get_eigen.argtypes = [C.c_void_p, C.c_int, _dp, _dp]
        for name in ("orc_forward_x", "orc_forward_y", "orc_inverse_y", "orc_inverse_x"):
            getattr(L, name).argtypes = [C.c_void_p, _dp, _dp]
            getattr(L, name).restype = None
        L.orc_thomas_z.argtypes = [C.c_void_p, _dp]
        L.orc_solve.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.orc_apply_operator_flux.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, C.c_double, _dp, _dp]
        L.orc_residual_norms.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, C.c_double, _dp, _dp, _dp]
        L.orc_dense_solve_3d.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, C.c_double, _dp, _dp]
        L.orc_plan_set_implicit_dirs.argtypes = [C.c_void_p, C.c_int]
        L.orc_apply_operator_flux_dirs.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, C.c_double, C.c_int,
                                                   _dp, _dp]
        L.orc_residual_norms_dirs.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, C.c_double, C.c_int, _dp,
                                              _dp, _dp]
        L.orc_dense_solve_3d_dirs.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, C.c_double, C.c_int, _dp,
                                              _dp]
        L.orc_divergence.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, _dp, _dp, _dp, C.c_double, _dp]
        L.orc_gradient.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _ip, _dp, _dp, _dp, _dp]
        L.orc_project.argtypes = [C.c_void_p, _dp, _dp, _dp, C.c_double, _dp, _dp, _dp, _dp, _dp, C.c_double, C.c_int]
        L.orc_num_threads.argtypes = []
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"oracle: {what} failed with status {rc}")


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _faces(xf):
    return np.ascontiguousarray(xf, dtype=np.float64)


def operator_1d(xf, bc):
    xf = _faces(xf)
    n = xf.size - 1
    w, a, b, c = (np.empty(n) for _ in range(4))
    _check(lib().orc_operator_1d(n, _ptr(xf), int(bc), _ptr(w), _ptr(a), _ptr(b), _ptr(c)), "operator_1d")
    return w, a, b, c


def symmetrize_1d(w, a, b, c):
    n = w.size
    d, o = np.empty(n), np.empty(n - 1)
    _check(lib().orc_symmetrize_1d(n, _ptr(w), _ptr(a), _ptr(b), _ptr(c), _ptr(d), _ptr(o)), "symmetrize_1d")
    return d, o


_eig_cache: dict = {}


def eig_1d(xf, bc, refine_steps: int = 2, cache: bool = True):
    """(lambda[n], qtilde[n,n]) with qtilde[i,m] = component i of mode m."""
    xf = _faces(xf)
    n = xf.size - 1
    key = (xf.tobytes(), int(bc), int(refine_steps))
    if cache and key in _eig_cache:
        return _eig_cache[key]
    lam, q = np.empty(n), np.empty((n, n))
    _check(lib().orc_eig_1d(n, _ptr(xf), int(bc), int(refine_steps), _ptr(lam), _ptr(q)), "eig_1d")
    if cache:
        _eig_cache[key] = (lam, q)
    return lam, q


class OraclePlan:
    """orc_plan handle.  Fields are numpy float64 arrays of shape (nz, ny, nx)."""

    def __init__(self, xf, yf, zf, bc, alpha: float = 0.0, refine_steps: int = 2, dirs: int = DIRS_XYZ):
        self.xf, self.yf, self.zf = _faces(xf), _faces(yf), _faces(zf)
        self.nx, self.ny, self.nz = self.xf.size - 1, self.yf.size - 1, self.zf.size - 1
        self.bc = tuple(int(b) for b in bc)
        self.alpha = float(alpha)
        lamx, qx = eig_1d(self.xf, self.bc[0], refine_steps)
        lamy, qy = eig_1d(self.yf, self.bc[1], refine_steps)
        h = C.c_void_p()
        _check(lib().orc_plan_create_with_eig(C.byref(h), self.nx, self.ny, self.nz, _ptr(self.xf), _ptr(self.yf),
                                              _ptr(self.zf), _bc(self.bc), self.alpha, _ptr(lamx), _ptr(qx),
                                              _ptr(lamy), _ptr(qy)), "plan_create")
        self._h = h
        self.dirs = int(dirs)
        if self.dirs != DIRS_XYZ:
            _check(lib().orc_plan_set_implicit_dirs(self._h, self.dirs), "plan_set_implicit_dirs")

    def close(self):
        if getattr(self, "_h", None):
            lib().orc_plan_destroy(self._h)
            self._h = None

    __del__ = close

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def singular(self) -> bool:
        return bool(lib().orc_plan_is_singular(self._h))

    def eigen(self, d: int):
        n = self.nx if d == 0 else self.ny
        lam, q = np.empty(n), np.empty((n, n))
        _check(lib().orc_plan_get_eigen(self._h, d, _ptr(lam), _ptr(q)), "get_eigen")
        return lam, q

    def _stage(self, name, x):
        x = np.ascontiguousarray(x, dtype=np.float64).reshape(self.shape)
        out = np.empty_like(x)
        getattr(lib(), name)(self._h, _ptr(x), _ptr(out))
        return out

    def forward_x(self, x):
        return self._stage("orc_forward_x", x)

    def forward_y(self, x):
        return self._stage("orc_forward_y", x)

    def inverse_y(self, x):
        return self._stage("orc_inverse_y", x)

    def inverse_x(self, x):
        return self._stage("orc_inverse_x", x)

    def thomas_z(self, x):
        out = np.array(x, dtype=np.float64, order="C").reshape(self.shape)
        _check(lib().orc_thomas_z(self._h, _ptr(out)), "thomas_z")
        return out

    def solve(self, f):
        f = np.ascontiguousarray(f, dtype=np.float64).reshape(self.shape)
        phi, work = np.empty_like(f), np.empty_like(f)
        _check(lib().orc_solve(self._h, _ptr(f), _ptr(phi), _ptr(work)), "solve")
        return phi


def apply_operator_flux(xf, yf, zf, bc, alpha, phi, dirs: int = DIRS_XYZ):
    xf, yf, zf = _faces(xf), _faces(yf), _faces(zf)
    nx, ny, nz = xf.size - 1, yf.size - 1, zf.size - 1
    phi = np.ascontiguousarray(phi, dtype=np.float64).reshape(nz, ny, nx)
    out = np.empty_like(phi)
    _check(lib().orc_apply_operator_flux_dirs(nx, ny, nz, _ptr(xf), _ptr(yf), _ptr(zf), _bc(bc), float(alpha),
                                              int(dirs), _ptr(phi), _ptr(out)), "apply_operator_flux")
    return out


def residual_norms(xf, yf, zf, bc, alpha, f, phi, dirs: int = DIRS_XYZ) -> dict:
    xf, yf, zf = _faces(xf), _faces(yf), _faces(zf)
    nx, ny, nz = xf.size - 1, yf.size - 1, zf.size - 1
    f = np.ascontiguousarray(f, dtype=np.float64).reshape(nz, ny, nx)
    phi = np.ascontiguousarray(phi, dtype=np.float64).reshape(nz, ny, nx)
    norms = np.empty(4)
    _check(lib().orc_residual_norms_dirs(nx, ny, nz, _ptr(xf), _ptr(yf), _ptr(zf), _bc(bc), float(alpha), int(dirs),
                                         _ptr(f), _ptr(phi), _ptr(norms)), "residual_norms")
    return {"rel2": norms[0], "relL2vol": norms[1], "relmax": norms[2], "backward": norms[3]}


def dense_solve_3d(xf, yf, zf, bc, alpha, f, dirs: int = DIRS_XYZ):
    xf, yf, zf = _faces(xf), _faces(yf), _faces(zf)
    nx, ny, nz = xf.size - 1, yf.size - 1, zf.size - 1
    f = np.ascontiguousarray(f, dtype=np.float64).reshape(nz, ny, nx)
    phi = np.empty_like(f)
    _check(lib().orc_dense_solve_3d_dirs(nx, ny, nz, _ptr(xf), _ptr(yf), _ptr(zf), _bc(bc), float(alpha), int(dirs),
                                         _ptr(f), _ptr(phi)), "dense_solve_3d")
    return phi


def face_shapes(nx, ny, nz):
    """Shapes of the staggered velocity arrays (reading A18): u on x-faces, v on y-faces, w on z-faces."""
    return (nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)


def divergence(xf, yf, zf, bc, u, v, w, scale: float = 1.0):
    xf, yf, zf = _faces(xf), _faces(yf), _faces(zf)
    nx, ny, nz = xf.size - 1, yf.size - 1, zf.size - 1
    su, sv, sw = face_shapes(nx, ny, nz)
    u = np.ascontiguousarray(u, dtype=np.float64).reshape(su)
    v = np.ascontiguousarray(v, dtype=np.float64).reshape(sv)
    w = np.ascontiguousarray(w, dtype=np.float64).reshape(sw)
    out = np.empty((nz, ny, nx))
    _check(lib().orc_divergence(nx, ny, nz, _ptr(xf), _ptr(yf), _ptr(zf), _bc(bc), _ptr(u), _ptr(v), _ptr(w),
                                float(scale), _ptr(out)), "divergence")
    return out


def gradient(xf, yf, zf, bc, phi):
    xf, yf, zf = _faces(xf), _faces(yf), _faces(zf)
    nx, ny, nz = xf.size - 1, yf.size - 1, zf.size - 1
    su, sv, sw = face_shapes(nx, ny, nz)
    phi = np.ascontiguousarray(phi, dtype=np.float64).reshape(nz, ny, nx)
    gu, gv, gw = np.empty(su), np.empty(sv), np.empty(sw)
    _check(lib().orc_gradient(nx, ny, nz, _ptr(xf), _ptr(yf), _ptr(zf), _bc(bc), _ptr(phi), _ptr(gu), _ptr(gv),
                              _ptr(gw)), "gradient")
    return gu, gv, gw


def project(plan: "OraclePlan", c: float, u, v, w, p=None, alpha_p: float = 0.0, dirs: int = DIRS_XYZ):
    """Eq. 2c-2e with the Poisson plan `plan`: returns (u, v, w, phi, p) as new arrays."""
    su, sv, sw = face_shapes(plan.nx, plan.ny, plan.nz)
    u = np.array(u, dtype=np.float64, order="C").reshape(su)
    v = np.array(v, dtype=np.float64, order="C").reshape(sv)
    w = np.array(w, dtype=np.float64, order="C").reshape(sw)
    phi = np.empty(plan.shape)
    pp = None if p is None else np.array(p, dtype=np.float64, order="C").reshape(plan.shape)
    _check(lib().orc_project(plan._h, _ptr(plan.xf), _ptr(plan.yf), _ptr(plan.zf), float(c), _ptr(u), _ptr(v), _ptr(w),
                             _ptr(phi), None if pp is None else _ptr(pp), float(alpha_p), int(dirs)), "project")
    return u, v, w, phi, pp
