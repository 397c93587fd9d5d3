"""ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front end of oracle/hard_oracle.cpp (the plain single-threaded fp64 C++ restatement of the
paper's explicit Euler finite-volume update) plus oracle/exact.py (exact
Riemann solution, Sedov-Taylor constant, the paper's L1 metric P:192-196).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
It imports nothing from paper_2509_08971_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hard_oracle.cpp")
_LIB = os.path.join(_HERE, "libhard_oracle.so")

SCHEME_A = 0  # WENO5-Z + HLL + Heun (paper)
SCHEME_B = 1  # MUSCL-minmod + HLLC + SSP-RK2 (north_star fallback)
BC_PERIODIC = 0
BC_OUTFLOW = 1
BC_REFLECT = 2   # reflecting wall (NEXT-2, G17)
ERR_NONPHYSICAL = -5

# -ffp-contract=off: no FMA contraction, so every operation rounds once in the order written.
CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared"]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", *CXXFLAGS, _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        vp = ctypes.c_void_p
        L.oracle_create.restype = vp
        L.oracle_create.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double, ctypes.c_int]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_set_spacing.argtypes = [vp] + [ctypes.c_double] * 3
        L.oracle_set_scheme.argtypes = [vp, ctypes.c_int]
        L.oracle_set_check.argtypes = [vp, ctypes.c_int]
        L.oracle_set_state.argtypes = [vp] + [dp] * 5
        L.oracle_get_state.argtypes = [vp] + [dp] * 5
        L.oracle_step.argtypes = [vp, ctypes.c_double, ctypes.c_int]
        L.oracle_step_dt.argtypes = [vp, ctypes.c_double, ctypes.c_int]
        L.oracle_max_dt.argtypes = [vp, dp]
        L.oracle_get_time.argtypes = [vp, dp, ctypes.POINTER(ctypes.c_longlong)]
        L.oracle_fallback_count.restype = ctypes.c_longlong
        L.oracle_fallback_count.argtypes = [vp]
        L.oracle_rhs.argtypes = [vp, dp]
        L.oracle_sum3sym.restype = ctypes.c_double
        L.oracle_sum3sym.argtypes = [ctypes.c_double] * 3
        L.oracle_wenoz.restype = ctypes.c_double
        L.oracle_wenoz.argtypes = [ctypes.c_double] * 5
        L.oracle_minmod.restype = ctypes.c_double
        L.oracle_minmod.argtypes = [ctypes.c_double] * 2
        L.oracle_cons_to_prim.restype = None
        L.oracle_cons_to_prim.argtypes = [dp, ctypes.c_double, dp]
        L.oracle_riemann.restype = None
        L.oracle_riemann.argtypes = [ctypes.c_int, dp, dp, ctypes.c_int, ctypes.c_double, dp]
        L.oracle_enable_radiation.argtypes = [vp]
        L.oracle_set_rad_energy.argtypes = [vp, dp]
        L.oracle_get_rad_energy.argtypes = [vp, dp]
        L.oracle_set_source.argtypes = [vp] + [ctypes.c_double] * 4
        L.oracle_rusanov.restype = ctypes.c_double
        L.oracle_rusanov.argtypes = [ctypes.c_double, ctypes.c_double, dp, dp, ctypes.c_int, ctypes.c_double]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__("oracle %s failed with code %d" % (what, code))
        self.code = code


class Oracle:
    """Same calls as the C-ABI of include/hard.h, with an oracle_ prefix underneath.

    State arrays are float64 numpy arrays of shape (nz, ny, nx) (x fastest), conserved variables
    (rho, mx, my, mz, E) of P:93 eq.2.
    """

    def __init__(self, nx, ny, nz, gamma, bc, scheme=SCHEME_A, spacing=None, check=True, radiation=False):
        self.L = lib()
        self.shape = (nz, ny, nx)
        self.h = self.L.oracle_create(nx, ny, nz, gamma, bc)
        if not self.h:
            raise OracleError(-1, "create")
        self._chk(self.L.oracle_set_scheme(self.h, scheme), "set_scheme")
        if spacing is not None:
            self._chk(self.L.oracle_set_spacing(self.h, *map(float, spacing)), "set_spacing")
        if radiation:
            self._chk(self.L.oracle_enable_radiation(self.h), "enable_radiation")
        if not check:
            self._chk(self.L.oracle_set_check(self.h, 0), "set_check")

    def _chk(self, rc, what):
        if rc != 0:
            raise OracleError(rc, what)

    def close(self):
        if self.h:
            self.L.oracle_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, rho, mx, my, mz, E):
        arrs = [np.ascontiguousarray(a, dtype=np.float64).reshape(self.shape) for a in (rho, mx, my, mz, E)]
        self._chk(self.L.oracle_set_state(self.h, *[_dp(a) for a in arrs]), "set_state")

    def get_state(self):
        out = [np.empty(self.shape, dtype=np.float64) for _ in range(5)]
        self._chk(self.L.oracle_get_state(self.h, *[_dp(a) for a in out]), "get_state")
        return out

    def set_rad_energy(self, er):
        a = np.ascontiguousarray(er, dtype=np.float64).reshape(self.shape)
        self._chk(self.L.oracle_set_rad_energy(self.h, _dp(a)), "set_rad_energy")

    def set_source(self, kappa, c_light, a_rad, cv):
        self._chk(self.L.oracle_set_source(self.h, float(kappa), float(c_light), float(a_rad), float(cv)), "set_source")

    def get_rad_energy(self):
        out = np.empty(self.shape, dtype=np.float64)
        self._chk(self.L.oracle_get_rad_energy(self.h, _dp(out)), "get_rad_energy")
        return out

    def step(self, cfl, nsteps=1):
        self._chk(self.L.oracle_step(self.h, float(cfl), int(nsteps)), "step")

    def step_dt(self, dt, nsteps=1):
        self._chk(self.L.oracle_step_dt(self.h, float(dt), int(nsteps)), "step_dt")

    def max_dt(self):
        v = ctypes.c_double()
        self._chk(self.L.oracle_max_dt(self.h, ctypes.byref(v)), "max_dt")
        return v.value

    def time(self):
        t = ctypes.c_double()
        n = ctypes.c_longlong()
        self._chk(self.L.oracle_get_time(self.h, ctypes.byref(t), ctypes.byref(n)), "get_time")
        return t.value, n.value

    def rhs(self, nf=5):
        """L(U) of the current state (eq.15): list of nf arrays of shape (nz, ny, nx)."""
        out = np.empty((nf,) + self.shape, dtype=np.float64)
        self._chk(self.L.oracle_rhs(self.h, _dp(out)), "rhs")
        return [out[f] for f in range(nf)]

    def fallbacks(self):
        return int(self.L.oracle_fallback_count(self.h))

    def run_to(self, t_end, cfl, max_steps=10 ** 7):
        """Harness loop of SURVEY §8(b): step(cfl) while t < t_end, clamping the last step."""
        n = 0
        while n < max_steps:
            t, _ = self.time()
            if t >= t_end:
                break
            dt = cfl * self.max_dt()
            if t + dt >= t_end:
                self.step_dt(t_end - t, 1)
                n += 1
                break
            self.step(cfl, 1)
            n += 1
        return n


def wenoz(a, b, c, d, e):
    return lib().oracle_wenoz(a, b, c, d, e)


def minmod(a, b):
    return lib().oracle_minmod(a, b)


def sum3sym(a, b, c):
    return lib().oracle_sum3sym(a, b, c)


def cons_to_prim(U, gamma):
    U = np.ascontiguousarray(U, dtype=np.float64)
    W = np.empty(5)
    lib().oracle_cons_to_prim(_dp(U), float(gamma), _dp(W))
    return W


def riemann(scheme, WL, WR, direction, gamma):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.empty(5)
    lib().oracle_riemann(int(scheme), _dp(WL), _dp(WR), int(direction), float(gamma), _dp(F))
    return F


def rusanov(EL, ER, WL, WR, direction, gamma):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    return lib().oracle_rusanov(float(EL), float(ER), _dp(WL), _dp(WR), int(direction), float(gamma))
