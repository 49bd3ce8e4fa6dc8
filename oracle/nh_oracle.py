"""ctypes wrapper of oracle/libnh_oracle.so (argument marshalling only; see nh_oracle.h)."""
from __future__ import annotations

import ctypes as C
import numpy as np

from . import build as _build


class _Params(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("tau", C.c_double), ("K", C.c_double), ("pitch", C.c_double),
                ("xi", C.c_double), ("gamma1", C.c_double), ("g", C.c_double * 3),
                ("anchoring", C.c_int), ("W0", C.c_double), ("fd_ratio", C.c_int),
                ("precision", C.c_int), ("coupling", C.c_int), ("alpha", C.c_double * 6),
                ("K3", C.c_double * 3)]


class OracleError(RuntimeError):
    pass


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        dp = C.POINTER(C.c_double)
        lib.nh_oracle_init_lattice.argtypes = [C.POINTER(_Params), C.POINTER(C.c_void_p)]
        lib.nh_oracle_set_director.argtypes = [C.c_void_p, dp]
        lib.nh_oracle_step.argtypes = [C.c_void_p, C.c_int, C.c_int]
        lib.nh_oracle_get_fields.argtypes = [C.c_void_p, dp, dp, dp, dp]
        lib.nh_oracle_get_populations.argtypes = [C.c_void_p, dp]
        lib.nh_oracle_set_velocity.argtypes = [C.c_void_p, dp]
        lib.nh_oracle_time.argtypes = [C.c_void_p]
        lib.nh_oracle_time.restype = C.c_long
        lib.nh_oracle_free.argtypes = [C.c_void_p]
        lib.nh_oracle_free.restype = None
        lib.nh_oracle_last_error.restype = C.c_char_p
        lib.nh_oracle_molecular_field.argtypes = [C.c_int] * 4 + [C.c_double] * 2 + [dp, dp]
        lib.nh_oracle_molecular_field_w0.argtypes = [C.c_int] * 4 + [C.c_double] * 3 + [dp, dp]
        lib.nh_oracle_director_rhs.argtypes = [C.c_int] * 4 + [C.c_double] * 4 + [dp, dp, dp]
        lib.nh_oracle_elastic_stress.argtypes = [C.c_int] * 4 + [C.c_double] * 2 + [dp, dp]
        lib.nh_oracle_elastic_force.argtypes = [C.c_int] * 4 + [C.c_double] * 2 + [dp, dp]
        lib.nh_oracle_frank3.argtypes = [C.c_int] * 4 + [dp, C.c_double, dp, dp, dp, dp]
        lib.nh_oracle_viscous_stress.argtypes = [C.c_int] * 4 + [C.c_double] * 4 + [dp, dp, dp, dp]
        lib.nh_oracle_lc_force.argtypes = [C.c_int] * 4 + [C.c_double] * 4 + [dp, dp, dp, dp]
        _lib = lib
    return _lib


def _check(rc):
    if rc != 0:
        raise OracleError("oracle error %d: %s" % (rc, _load().nh_oracle_last_error().decode()))


def _ptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a, shape):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.shape != shape:
        raise ValueError("expected shape %r, got %r" % (shape, a.shape))
    return a


def num_threads() -> int:
    return int(_load().nh_oracle_num_threads())


class Oracle:
    """One oracle lattice; same call surface as the CUDA binding (init / set_director / step / get_fields)."""

    def __init__(self, nx, ny, nz, tau, K=0.0, pitch=0.0, xi=0.0, gamma1=1.0, g=(0.0, 0.0, 0.0),
                 anchoring=0, W0=0.0, fd_ratio=1, precision=0, coupling=3, alpha=(0.0,) * 6, K3=(0.0, 0.0, 0.0), **_ignored):
        lib = _load()
        self.p = _Params(nx, ny, nz, tau, K, pitch, xi, gamma1, (C.c_double * 3)(*g), anchoring, W0,
                         fd_ratio, precision, coupling, (C.c_double * 6)(*alpha), (C.c_double * 3)(*K3))
        self.shape = (nz, ny, nx)
        self._h = C.c_void_p()
        _check(lib.nh_oracle_init_lattice(C.byref(self.p), C.byref(self._h)))

    def __del__(self):
        if getattr(self, "_h", None) and self._h.value:
            _load().nh_oracle_free(self._h)
            self._h = None

    def set_director(self, n):
        n = _f64(n, (3,) + self.shape)
        _check(_load().nh_oracle_set_director(self._h, _ptr(n)))

    def set_velocity(self, u):
        """Test-only: populations := equilibrium(rho = 1, u) on fluid cells."""
        u = _f64(u, (3,) + self.shape)
        _check(_load().nh_oracle_set_velocity(self._h, _ptr(u)))

    def step(self, n_lb, n_fd=-1):
        _check(_load().nh_oracle_step(self._h, int(n_lb), int(n_fd)))

    @property
    def time(self):
        return int(_load().nh_oracle_time(self._h))

    def get_fields(self):
        rho = np.empty(self.shape)
        u = np.empty((3,) + self.shape)
        n = np.empty((3,) + self.shape)
        F = np.empty((3,) + self.shape)
        _check(_load().nh_oracle_get_fields(self._h, _ptr(rho), _ptr(u), _ptr(n), _ptr(F)))
        return dict(rho=rho, u=u, n=n, F=F)

    def get_populations(self):
        f = np.empty((19,) + self.shape)
        _check(_load().nh_oracle_get_populations(self._h, _ptr(f)))
        return f


def _dims(n):
    _, nz, ny, nx = n.shape
    return nx, ny, nz


def molecular_field(n, K, q0, periodic_z=False, W0=0.0):
    n = np.ascontiguousarray(n, dtype=np.float64)
    h = np.empty_like(n)
    nx, ny, nz = _dims(n)
    if W0:
        _check(_load().nh_oracle_molecular_field_w0(nx, ny, nz, int(periodic_z), K, q0, W0, _ptr(n), _ptr(h)))
    else:
        _check(_load().nh_oracle_molecular_field(nx, ny, nz, int(periodic_z), K, q0, _ptr(n), _ptr(h)))
    return h


def director_rhs(n, u, K, q0, xi, gamma1, periodic_z=False):
    n = np.ascontiguousarray(n, dtype=np.float64)
    u = _f64(u, n.shape)
    R = np.empty_like(n)
    nx, ny, nz = _dims(n)
    _check(_load().nh_oracle_director_rhs(nx, ny, nz, int(periodic_z), K, q0, xi, gamma1,
                                          _ptr(n), _ptr(u), _ptr(R)))
    return R


def elastic_stress(n, K, q0, periodic_z=False):
    n = np.ascontiguousarray(n, dtype=np.float64)
    nx, ny, nz = _dims(n)
    s = np.empty((9, nz, ny, nx))
    _check(_load().nh_oracle_elastic_stress(nx, ny, nz, int(periodic_z), K, q0, _ptr(n), _ptr(s)))
    return s.reshape(3, 3, nz, ny, nx)


def elastic_force(n, K, q0, periodic_z=False):
    n = np.ascontiguousarray(n, dtype=np.float64)
    F = np.empty_like(n)
    nx, ny, nz = _dims(n)
    _check(_load().nh_oracle_elastic_force(nx, ny, nz, int(periodic_z), K, q0, _ptr(n), _ptr(F)))
    return F


def viscous_stress(n, u, K, q0, xi, gamma1, alpha, periodic_z=False):
    """Leslie viscous stress (Eq. 3 with alpha4', N from Eq. 9); alpha = (a1, a2, a3, a4', a5, a6)."""
    n = np.ascontiguousarray(n, dtype=np.float64)
    u = _f64(u, n.shape)
    al = np.ascontiguousarray(alpha, dtype=np.float64)
    nx, ny, nz = _dims(n)
    s = np.empty((9, nz, ny, nx))
    _check(_load().nh_oracle_viscous_stress(nx, ny, nz, int(periodic_z), K, q0, xi, gamma1, _ptr(al),
                                            _ptr(n), _ptr(u), _ptr(s)))
    return s.reshape(3, 3, nz, ny, nx)


def lc_force(n, u, K, q0, xi, gamma1, alpha, periodic_z=False):
    """F^LC = d_b (sigma^e + sigma^v)_ab, Eq. 12."""
    n = np.ascontiguousarray(n, dtype=np.float64)
    u = _f64(u, n.shape)
    al = np.ascontiguousarray(alpha, dtype=np.float64)
    F = np.empty_like(n)
    nx, ny, nz = _dims(n)
    _check(_load().nh_oracle_lc_force(nx, ny, nz, int(periodic_z), K, q0, xi, gamma1, _ptr(al),
                                      _ptr(n), _ptr(u), _ptr(F)))
    return F


def frank3(n, K3, q0, periodic_z=False):
    """Three-constant Frank energy (Eqs. 7-8): returns (h [3,...], sigma [3,3,...], total energy)."""
    n = np.ascontiguousarray(n, dtype=np.float64)
    k3 = np.ascontiguousarray(K3, dtype=np.float64)
    nx, ny, nz = _dims(n)
    h = np.empty_like(n)
    s = np.empty((9, nz, ny, nx))
    e = C.c_double(0.0)
    _check(_load().nh_oracle_frank3(nx, ny, nz, int(periodic_z), _ptr(k3), q0, _ptr(n), _ptr(h), _ptr(s),
                                    C.cast(C.byref(e), C.POINTER(C.c_double))))
    return h, s.reshape(3, 3, nz, ny, nx), e.value
