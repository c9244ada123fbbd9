"""accLB CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front-end of ``oracle/acclb_oracle.c`` (plain C, fp64, paper-literal two-pass step of
arXiv 2505.01126; see that file's header).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports
nothing from ``paper_2505_01126_b200`` and that package imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "acclb_oracle.c"
_LIB = _HERE / "libacclb_oracle.so"


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2 -fopenmp -ffp-contract=off).  Building the checker is not using it."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class OracleParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("tau", C.c_double),
        ("two_phase", C.c_int),
        ("rho_l", C.c_double), ("rho_g", C.c_double), ("sigma", C.c_double),
        ("mobility", C.c_double), ("width", C.c_double),
        ("force_type", C.c_int), ("force_amp", C.c_double), ("force_k", C.c_int),
        ("force_period", C.c_int * 3), ("force_origin", C.c_int * 3),
        ("gravity", C.c_double * 3), ("rho_ref", C.c_double), ("phi_rk3", C.c_int),
    ]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [C.POINTER(OracleParams)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_init.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.oracle_step.argtypes = [C.c_void_p, C.c_int]
        L.oracle_moments.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.oracle_diagnostics.argtypes = [C.c_void_p, _dp, C.c_int]
        L.oracle_get_populations.argtypes = [C.c_void_p, _dp]
        L.oracle_set_populations.argtypes = [C.c_void_p, _dp]
        L.oracle_get_hermite.argtypes = [C.c_void_p, _dp]
        L.oracle_get_accel.argtypes = [C.c_void_p, _dp]
        L.oracle_lattice.argtypes = [C.POINTER(C.c_int), _dp]
        L.oracle_feq.argtypes = [C.c_double, _dp, _dp]
        L.oracle_guo.argtypes = [_dp, _dp, _dp]
        L.oracle_fneq.argtypes = [_dp, _dp]
        L.oracle_weno5.restype = C.c_double
        L.oracle_weno5.argtypes = [C.c_double] * 5
        L.oracle_gradient.argtypes = [_dp, C.c_int, C.c_int, C.c_int, _dp]
        L.oracle_laplacian.argtypes = [_dp, C.c_int, C.c_int, C.c_int, _dp]
        L.oracle_body_force.argtypes = [C.POINTER(OracleParams), C.c_int, C.c_int, C.c_int, _dp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


DIAG_NAMES = ("ke", "dissipation", "sum_phi", "sum_pstar", "sum_mx", "sum_my", "sum_mz", "umax", "step")


class Oracle:
    """One periodic box.  Fields are numpy fp64, scalars [nz][ny][nx] (x fastest), vectors [3][nz][ny][nx]."""

    def __init__(self, nx, ny, nz, *, tau, two_phase=False, rho_l=1.0, rho_g=1.0, sigma=0.0, mobility=0.0,
                 width=4.0, force_type=0, force_amp=0.0, force_k=1, force_period=(0, 0, 0),
                 force_origin=(0, 0, 0), gravity=(0.0, 0.0, 0.0), rho_ref=0.0, phi_rk3=0):
        self.params = OracleParams(nx, ny, nz, tau, int(two_phase), rho_l, rho_g, sigma, mobility, width,
                                   force_type, force_amp, force_k,
                                   (C.c_int * 3)(*force_period), (C.c_int * 3)(*force_origin),
                                   (C.c_double * 3)(*gravity), rho_ref, int(phi_rk3))
        self.shape = (nz, ny, nx)
        self.n = nx * ny * nz
        self.two_phase = bool(two_phase)
        self._h = lib().oracle_create(C.byref(self.params))
        if not self._h:
            raise ValueError("oracle_create failed (bad parameters or out of memory)")

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def init(self, rho, u, phi=None):
        rho = _c(rho, self.shape)
        u = _c(u, (3,) + self.shape)
        phi = _c(phi, self.shape) if phi is not None else None
        if lib().oracle_init(self._h, _p(rho), _p(u), _p(phi)) != 0:
            raise ValueError("oracle_init failed")

    def step(self, nsteps=1):
        if lib().oracle_step(self._h, int(nsteps)) != 0:
            raise ValueError("oracle_step failed")

    def moments(self):
        rho = np.empty(self.shape)
        u = np.empty((3,) + self.shape)
        phi = np.empty(self.shape) if self.two_phase else None
        lib().oracle_moments(self._h, _p(rho), _p(u), _p(phi))
        return rho, u, phi

    def diagnostics(self):
        out = np.zeros(9)
        if lib().oracle_diagnostics(self._h, _p(out), 9) != 0:
            raise ValueError("oracle_diagnostics failed")
        return dict(zip(DIAG_NAMES, out.tolist()))

    # raw access for the pin tests
    def populations(self):
        f = np.empty((27,) + self.shape)
        lib().oracle_get_populations(self._h, _p(f))
        return f

    def set_populations(self, f):
        f = _c(f, (27,) + self.shape)
        lib().oracle_set_populations(self._h, _p(f))

    def hermite(self):
        """a_ab (xx,yy,zz,xy,xz,yz) as left by the last moments()/diagnostics() call."""
        a = np.empty((6,) + self.shape)
        lib().oracle_get_hermite(self._h, _p(a))
        return a

    def accel(self):
        A = np.empty((3,) + self.shape)
        lib().oracle_get_accel(self._h, _p(A))
        return A


def lattice():
    c = (C.c_int * 81)()
    w = np.empty(27)
    lib().oracle_lattice(c, _p(w))
    return np.array(list(c), dtype=np.int64).reshape(27, 3), w


def feq(pstar, u):
    out = np.empty(27)
    u = _c(u, (3,))
    lib().oracle_feq(float(pstar), _p(u), _p(out))
    return out


def guo(u, A):
    out = np.empty(27)
    u, A = _c(u, (3,)), _c(A, (3,))
    lib().oracle_guo(_p(u), _p(A), _p(out))
    return out


def fneq(a6):
    out = np.empty(27)
    a6 = _c(a6, (6,))
    lib().oracle_fneq(_p(a6), _p(out))
    return out


def weno5(a, b, c, d, e):
    return lib().oracle_weno5(a, b, c, d, e)


def gradient(psi):
    psi = _c(psi)
    nz, ny, nx = psi.shape
    out = np.empty((3, nz, ny, nx))
    lib().oracle_gradient(_p(psi), nx, ny, nz, _p(out))
    return out


def laplacian(psi):
    psi = _c(psi)
    nz, ny, nx = psi.shape
    out = np.empty((nz, ny, nx))
    lib().oracle_laplacian(_p(psi), nx, ny, nz, _p(out))
    return out


def body_force(params: OracleParams, x, y, z):
    out = np.empty(3)
    lib().oracle_body_force(C.byref(params), x, y, z, _p(out))
    return out
