"""CPU oracle for the CLTx hot path (arxiv 1812.00525, section 2) -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares no code with ``paper_1812_00525_b200`` (the CUDA path) and
imports nothing from it.  The arithmetic lives in ``clt_oracle.c`` (plain C, FP64, gcc
``-O2 -ffp-contract=off``); this module only builds it and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "clt_oracle.c")
_LIB = os.path.join(_HERE, "libclt_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile clt_oracle.c -> libclt_oracle.so (in-tree).  No fast-math, no FMA contraction (hazard H3)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
               "-std=c11", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_dp = ctypes.POINTER(ctypes.c_double)


def _ptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def lib():
    global _lib
    with _lock:
        if _lib is None:
            L = ctypes.CDLL(build())
            L.oracle_create.restype = ctypes.c_void_p
            L.oracle_create.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 11
            L.oracle_destroy.argtypes = [ctypes.c_void_p]
            L.oracle_set_dt.argtypes = [ctypes.c_void_p, ctypes.c_double]
            L.oracle_set_equilibrium.argtypes = [ctypes.c_void_p, _dp]
            L.oracle_set_state.argtypes = [ctypes.c_void_p, _dp]
            L.oracle_get_state.argtypes = [ctypes.c_void_p, _dp]
            L.oracle_get_step.restype = ctypes.c_int64
            L.oracle_get_step.argtypes = [ctypes.c_void_p]
            L.oracle_get_time.restype = ctypes.c_double
            L.oracle_get_time.argtypes = [ctypes.c_void_p]
            L.oracle_curl_J1.argtypes = [ctypes.c_void_p, _dp, _dp]
            L.oracle_E1.argtypes = [ctypes.c_void_p, _dp, _dp]
            L.oracle_hall_G.argtypes = [ctypes.c_void_p, _dp, _dp]
            L.oracle_set_hall.argtypes = [ctypes.c_void_p, ctypes.c_double]
            L.oracle_set_phi_scheme.argtypes = [ctypes.c_void_p, ctypes.c_int]
            L.oracle_rhs_of.argtypes = [ctypes.c_void_p, _dp, _dp]
            L.oracle_rhs.argtypes = [ctypes.c_void_p, _dp]
            L.oracle_step.argtypes = [ctypes.c_void_p, ctypes.c_int]
            L.oracle_step_cfl.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double]
            L.oracle_get_dt.restype = ctypes.c_double
            L.oracle_get_dt.argtypes = [ctypes.c_void_p]
            L.oracle_diagnostics.argtypes = [ctypes.c_void_p, _dp]
            L.oracle_divB.argtypes = [ctypes.c_void_p, _dp, _dp]
            L.oracle_setdt.restype = ctypes.c_double
            L.oracle_setdt.argtypes = [ctypes.c_void_p, ctypes.c_double]
            L.oracle_apply_scalar_op.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, _dp]
            L.oracle_apply_vector_op.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, _dp]
            L.oracle_rk4.argtypes = [ctypes.c_size_t, _dp, ctypes.c_double, ctypes.c_int, RHS_FN,
                                     ctypes.c_void_p, _dp, _dp, _dp, _dp, _dp]
            _lib = L
    return _lib


RHS_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, _dp, _dp)

SCALAR_OPS = {"d1R": 0, "d1P": 1, "d1Z": 2, "d2R": 3, "d2P": 4, "d2Z": 5, "d1R_Rf": 6,
              "laplacian": 7, "divergence": 8, "div_c": 9}
VECTOR_OPS = {"grad": 0, "curl_c": 1, "vector_laplacian": 2, "advect_vector": 3}
DIAG_NAMES = ("kinetic", "magnetic", "magnetic_pert", "magnetic_n1", "max_divB")


class Oracle:
    """One oracle context: grid + physics parameters, equilibrium, state.

    Arrays are numpy float64, C-contiguous, shaped ``[8, nphi, nZ, nR]`` (state), ``[8, nZ, nR]``
    (equilibrium), ``[3, nphi, nZ, nR]`` (vector fields), ``[nphi, nZ, nR]`` (scalars).
    """

    def __init__(self, nR, nphi, nZ, Rmin, Rmax, Zmin, Zmax, phi_extent=0.0, gamma=5.0 / 3.0, eta=0.0, nu=0.0,
                 D=0.0, kappa=0.0, dt=0.0, d_i=0.0, phi_scheme=0):
        self.L = lib()
        self.nR, self.nphi, self.nZ = int(nR), int(nphi), int(nZ)
        self.h = self.L.oracle_create(self.nR, self.nphi, self.nZ, Rmin, Rmax, Zmin, Zmax, phi_extent, gamma, eta,
                                      nu, D, kappa, dt)
        if not self.h:
            raise ValueError("oracle_create rejected the grid")
        self.shape = (self.nphi, self.nZ, self.nR)
        self.L.oracle_set_equilibrium(self.h, None)
        if d_i:
            self.L.oracle_set_hall(self.h, float(d_i))
        if phi_scheme:
            self.L.oracle_set_phi_scheme(self.h, int(phi_scheme))

    def close(self):
        if getattr(self, "h", None):
            self.L.oracle_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, a, lead):
        a = np.ascontiguousarray(a, dtype=np.float64)
        want = (lead,) + self.shape if lead else self.shape
        assert a.shape == want, (a.shape, want)
        return a

    def set_dt(self, dt):
        self.L.oracle_set_dt(self.h, float(dt))

    def set_equilibrium(self, U0):
        if U0 is None:
            self.L.oracle_set_equilibrium(self.h, None)
            return
        U0 = np.ascontiguousarray(U0, dtype=np.float64)
        assert U0.shape == (8, self.nZ, self.nR)
        self.L.oracle_set_equilibrium(self.h, _ptr(U0))

    def set_state(self, U):
        self.L.oracle_set_state(self.h, _ptr(self._chk(U, 8)))

    def get_state(self):
        U = np.empty((8,) + self.shape)
        self.L.oracle_get_state(self.h, _ptr(U))
        return U

    @property
    def step_count(self):
        return int(self.L.oracle_get_step(self.h))

    @property
    def time(self):
        return float(self.L.oracle_get_time(self.h))

    def curl_J1(self, U):
        out = np.empty((3,) + self.shape)
        self.L.oracle_curl_J1(self.h, _ptr(self._chk(U, 8)), _ptr(out))
        return out

    def E1(self, U):
        out = np.empty((3,) + self.shape)
        self.L.oracle_E1(self.h, _ptr(self._chk(U, 8)), _ptr(out))
        return out

    def hall_G(self, U):
        out = np.empty((3,) + self.shape)
        self.L.oracle_hall_G(self.h, _ptr(self._chk(U, 8)), _ptr(out))
        return out

    def set_hall(self, d_i):
        self.L.oracle_set_hall(self.h, float(d_i))

    def set_phi_scheme(self, scheme):
        """0 = 4th-order finite differences in phi, 1 = pseudo-spectral."""
        self.L.oracle_set_phi_scheme(self.h, int(scheme))

    def rhs_of(self, U):
        K = np.empty((8,) + self.shape)
        self.L.oracle_rhs_of(self.h, _ptr(self._chk(U, 8)), _ptr(K))
        return K

    def rhs(self):
        K = np.empty((8,) + self.shape)
        self.L.oracle_rhs(self.h, _ptr(K))
        return K

    def step(self, n=1):
        self.L.oracle_step(self.h, int(n))

    def step_cfl(self, n, cfl):
        """n RK4 steps, each with dt = SETDT(cfl) of the state at its start (Fig. 3-4)."""
        self.L.oracle_step_cfl(self.h, int(n), float(cfl))

    @property
    def dt(self):
        return float(self.L.oracle_get_dt(self.h))

    def diagnostics(self):
        out = np.empty(5)
        self.L.oracle_diagnostics(self.h, _ptr(out))
        return dict(zip(DIAG_NAMES, out.tolist()))

    def divB(self, U):
        out = np.empty(self.shape)
        self.L.oracle_divB(self.h, _ptr(self._chk(U, 8)), _ptr(out))
        return out

    def setdt(self, cfl):
        return float(self.L.oracle_setdt(self.h, float(cfl)))

    def scalar_op(self, name, f):
        which = SCALAR_OPS[name]
        f = self._chk(f, 3 if which >= 8 else 0)
        out = np.empty(self.shape)
        self.L.oracle_apply_scalar_op(self.h, which, _ptr(f), _ptr(out))
        return out

    def vector_op(self, name, f):
        which = VECTOR_OPS[name]
        f = self._chk(f, {0: 0, 1: 3, 2: 3, 3: 6}[which])
        out = np.empty((3,) + self.shape)
        self.L.oracle_apply_vector_op(self.h, which, _ptr(f), _ptr(out))
        return out


def rk4(U, dt, nsteps, rhs):
    """Run the oracle's RK4 routine on a flat float64 vector with a Python RHS ``rhs(U) -> K`` (pin P8)."""
    U = np.ascontiguousarray(U, dtype=np.float64).copy()
    n = U.size

    def thunk(_user, pU, pK):
        u = np.ctypeslib.as_array(pU, shape=(n,))
        k = np.ctypeslib.as_array(pK, shape=(n,))
        k[:] = rhs(u)

    cb = RHS_FN(thunk)
    work = [np.zeros(n) for _ in range(5)]
    lib().oracle_rk4(n, _ptr(U), float(dt), int(nsteps), cb, None, *[_ptr(w) for w in work])
    return U
