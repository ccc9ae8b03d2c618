"""CPU ORACLE -- TEST INFRASTRUCTURE ONLY (see clvisc_oracle.cpp header).

ctypes binding of the plain fp64 C++ oracle.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package; the product
(the CUDA package) never does.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "clvisc_oracle.cpp")
_LIB = os.path.join(_HERE, "libclvisc_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, no FMA contraction, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fPIC",
                               "-shared", "-o", _LIB, _SRC])
    return _LIB


def _bind(path):
    """dlopen one build of the oracle and declare its C ABI."""
    lib = ctypes.CDLL(path)
    dp = ctypes.POINTER(ctypes.c_double)
    ip = ctypes.POINTER(ctypes.c_int)
    lib.oracle_create.restype = ctypes.c_void_p
    lib.oracle_create.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [ip, ctypes.c_int,
                                  ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                  ctypes.c_double, ctypes.c_double, dp, dp, ctypes.c_double,
                                  ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                  ctypes.c_double, ctypes.c_double, ctypes.c_int]
    lib.oracle_destroy.argtypes = [ctypes.c_void_p]
    for name, nptr in [("oracle_load", 2), ("oracle_set_history", 1), ("oracle_read", 3),
                       ("oracle_read_T", 1), ("oracle_read_history", 1), ("oracle_diag", 1),
                       ("oracle_set_state", 3), ("oracle_load_ext", 4), ("oracle_read_ext", 2),
                       ("oracle_set_ext", 2)]:
        f = getattr(lib, name)
        f.restype = ctypes.c_int
        f.argtypes = [ctypes.c_void_p] + [dp] * nptr
    lib.oracle_step.restype = ctypes.c_int
    lib.oracle_step.argtypes = [ctypes.c_void_p, ctypes.c_int]
    lib.oracle_rhs.restype = ctypes.c_int
    lib.oracle_rhs.argtypes = [ctypes.c_void_p, dp, ctypes.c_double, dp, dp]
    lib.oracle_eos.argtypes = [ctypes.c_void_p, ctypes.c_double, dp]
    lib.oracle_rootfind.argtypes = [ctypes.c_void_p, dp, dp]
    lib.oracle_limit_pi.restype = ctypes.c_int
    lib.oracle_limit_pi.argtypes = [ctypes.c_void_p, ctypes.c_double, dp]
    lib.oracle_set_option.restype = ctypes.c_int
    lib.oracle_set_option.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double]
    return lib


def _load():
    global _lib
    if _lib is None:
        _lib = _bind(build())
    return _lib


def build_variant(out_path: str, extra_flags=()):
    """A second build of the SAME source with different compiler flags (e.g. -ffp-contract=fast), used by the tests
    that measure how far two correct roundings of the oracle drift apart.  Returns a library handle for
    Oracle(..., lib=handle)."""
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared"] + list(extra_flags) + ["-o", out_path, _SRC]
    subprocess.check_call(cmd)
    return _bind(out_path)


def _p(a):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


class Oracle:
    """fp64 CPU oracle of the KT-RK2 viscous hydro step; same call shapes as the hydro_* C ABI."""

    def __init__(self, nx, ny, nz, dx, dy, deta, dtau, tau0, eos, eta_over_s, bc=(0, 0, 0),
                 geometry=0, minmod_theta=1.1, e_floor=1e-7, pi_limit_xi=1.0, v_max=0.999,
                 strict_eq53=0, lib=None):
        lib = self._lib = lib if lib is not None else _load()
        self.shape = (nz, ny, nx)
        self.N = nx * ny * nz
        bca = (ctypes.c_int * 3)(*bc)
        P = None if eos["P"] is None else np.ascontiguousarray(eos["P"], dtype=np.float64)
        T = None if eos["T"] is None else np.ascontiguousarray(eos["T"], dtype=np.float64)
        self._h = lib.oracle_create(nx, ny, nz, dx, dy, deta, bca, geometry, dtau, tau0,
                                    int(eos["kind"]), int(eos["n"]), float(eos["e_min"]),
                                    float(eos["e_max"]), _p(P), _p(T), float(eos["c_sb"]),
                                    float(eta_over_s), minmod_theta, e_floor, pi_limit_xi, v_max,
                                    strict_eq53)
        if not self._h:
            raise ValueError("oracle_create: invalid arguments")
        self.viscous = eta_over_s > 0

    def __del__(self):
        if getattr(self, "_h", None):
            self._lib.oracle_destroy(self._h)
            self._h = None

    def load(self, T, pi=None):
        T = np.ascontiguousarray(T, dtype=np.float64).reshape(4, -1)
        pi = None if pi is None else np.ascontiguousarray(pi, dtype=np.float64).reshape(10, -1)
        assert T.shape[1] == self.N
        return self._lib.oracle_load(self._h, _p(T), _p(pi))

    def set_state(self, e, u3, pi=None):
        e = np.ascontiguousarray(e, dtype=np.float64).reshape(-1)
        u3 = np.ascontiguousarray(u3, dtype=np.float64).reshape(3, -1)
        pi = None if pi is None else np.ascontiguousarray(pi, dtype=np.float64).reshape(10, -1)
        return self._lib.oracle_set_state(self._h, _p(e), _p(u3), _p(pi))

    def set_history(self, uprev3):
        a = np.ascontiguousarray(uprev3, dtype=np.float64).reshape(3, -1)
        return self._lib.oracle_set_history(self._h, _p(a))

    def step(self, n=1):
        rc = self._lib.oracle_step(self._h, int(n))
        if rc:
            raise RuntimeError(f"oracle_step rc={rc}")

    def read(self):
        e = np.empty(self.N)
        u = np.empty((4, self.N))
        pi = np.empty((10, self.N))
        self._lib.oracle_read(self._h, _p(e), _p(u), _p(pi))
        return e.reshape(self.shape), u.reshape((4,) + self.shape), pi.reshape((10,) + self.shape)

    def read_T(self):
        T = np.empty((4, self.N))
        self._lib.oracle_read_T(self._h, _p(T))
        return T.reshape((4,) + self.shape)

    def read_history(self):
        u = np.empty((3, self.N))
        self._lib.oracle_read_history(self._h, _p(u))
        return u.reshape((3,) + self.shape)

    def diag(self):
        d = np.zeros(9)
        self._lib.oracle_diag(self._h, _p(d))
        return dict(tau=d[0], step=int(d[1]), cfl=tuple(d[2:5]), e_max=d[5], floored=int(d[6]),
                    clamped=int(d[7]), pi_limited=int(d[8]))

    def rhs(self, dtu4, tau):
        dtu4 = np.ascontiguousarray(dtu4, dtype=np.float64).reshape(4, -1)
        ST = np.zeros((4, self.N))
        SP = np.zeros((10, self.N))
        self._lib.oracle_rhs(self._h, _p(dtu4), float(tau), _p(ST), _p(SP))
        return ST.reshape((4,) + self.shape), SP.reshape((10,) + self.shape)

    def eos(self, e):
        out = np.zeros(3)
        self._lib.oracle_eos(self._h, float(e), _p(out))
        return tuple(out)

    def limit_pi(self, e, pi10):
        """pi limiter (A14) on one cell: returns (scaled pi[10], acted?)."""
        p = np.array(pi10, dtype=np.float64)
        acted = self._lib.oracle_limit_pi(self._h, float(e), _p(p))
        return p, bool(acted)

    OPT_HEUN_PRINTED, OPT_LAMBDA1_HAT, OPT_C_TAU, OPT_EXT, OPT_ZETA_S = 0, 1, 2, 3, 4

    # -- bulk pressure Pi and net-baryon density n (after set_option(OPT_EXT, 1)) -------------
    def load_ext(self, T, pi=None, Pi=None, nb=None):
        T = np.ascontiguousarray(T, dtype=np.float64).reshape(4, -1)
        pi = None if pi is None else np.ascontiguousarray(pi, dtype=np.float64).reshape(10, -1)
        Pi = None if Pi is None else np.ascontiguousarray(Pi, dtype=np.float64).reshape(-1)
        nb = None if nb is None else np.ascontiguousarray(nb, dtype=np.float64).reshape(-1)
        return self._lib.oracle_load_ext(self._h, _p(T), _p(pi), _p(Pi), _p(nb))

    def set_ext(self, Pi=None, nb=None):
        Pi = None if Pi is None else np.ascontiguousarray(Pi, dtype=np.float64).reshape(-1)
        nb = None if nb is None else np.ascontiguousarray(nb, dtype=np.float64).reshape(-1)
        if self._lib.oracle_set_ext(self._h, _p(Pi), _p(nb)):
            raise ValueError("oracle_set_ext: the extension is off (set_option(OPT_EXT, 1) on a viscous run)")

    def read_ext(self):
        Pi, nb = np.empty(self.N), np.empty(self.N)
        self._lib.oracle_read_ext(self._h, _p(Pi), _p(nb))
        return Pi.reshape(self.shape), nb.reshape(self.shape)

    def set_option(self, key, value):
        if self._lib.oracle_set_option(self._h, int(key), float(value)):
            raise ValueError("oracle_set_option: unknown key")

    def rootfind(self, M4):
        M4 = np.ascontiguousarray(M4, dtype=np.float64)
        out = np.zeros(4)
        self._lib.oracle_rootfind(self._h, _p(M4), _p(out))
        return out
