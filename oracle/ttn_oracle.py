"""ctypes binding of oracle/ttn_oracle.c -- TEST INFRASTRUCTURE ONLY (see the C header).

The oracle is plain C built with gcc; this module compiles it on first use (or when the
source is newer than the shared object) and marshals numpy arrays.  Couplings are widened
to float64 here: the CUDA path receives the same values as float32 data.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ttn_oracle.c")
_SO = os.path.join(_HERE, "libttn_oracle.so")
_lib = None


class OracleOverflow(ArithmeticError):
    """A 128-bit degeneracy count overflowed (checked addition)."""


def build(force: bool = False) -> str:
    """Compile ttn_oracle.c -> libttn_oracle.so with gcc (OpenMP)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        u64p = ctypes.POINTER(ctypes.c_uint64)
        i8p = ctypes.POINTER(ctypes.c_int8)
        lib.ttn_oracle_brute_ising.argtypes = [ctypes.c_int, dp, dp, dp, dp, u64p, i8p]
        lib.ttn_oracle_brute_potts3.argtypes = [ctypes.c_int, dp, dp, dp, u64p, i8p]
        lib.ttn_oracle_dp_ising.argtypes = [ctypes.c_int, dp, dp, dp, ctypes.c_int, ctypes.c_int,
                                            dp, u64p, u64p, i8p]
        lib.ttn_oracle_dp_potts3.argtypes = [ctypes.c_int, dp, dp, ctypes.c_int, ctypes.c_int,
                                             dp, u64p, u64p, i8p]
        lib.ttn_oracle_ising_energy.argtypes = [ctypes.c_int, dp, dp, dp, i8p]
        lib.ttn_oracle_ising_energy.restype = ctypes.c_double
        lib.ttn_oracle_potts3_energy.argtypes = [ctypes.c_int, dp, dp, i8p]
        lib.ttn_oracle_potts3_energy.restype = ctypes.c_double
        lib.ttn_oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _f64(a, n, name):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1))
    if a.size != n:
        raise ValueError(f"{name}: expected {n} values, got {a.size}")
    if n == 0:  # L = 1: no bonds; hand C a valid (never read) pointer
        a = np.zeros(1, dtype=np.float64)
    return a


def _ptr(a, ty):
    return a.ctypes.data_as(ctypes.POINTER(ty)) if a is not None else None


def _check(rc):
    if rc == 2:
        raise OracleOverflow("128-bit degeneracy overflow")
    if rc != 0:
        raise RuntimeError(f"oracle error {rc}")


def num_threads() -> int:
    return int(_load().ttn_oracle_num_threads())


def _ising_args(L, Jh, Jv, h):
    Jh = _f64(Jh, L * (L - 1), "Jh")
    Jv = _f64(Jv, (L - 1) * L, "Jv")
    h = _f64(h, L * L, "h") if h is not None else None
    return Jh, Jv, h


def brute_ising(L, Jh, Jv, h=None):
    """Definition of E0, g, sigma* by enumeration (Eq. (1)). Returns (E0, g, sigma[L,L])."""
    Jh, Jv, h = _ising_args(L, Jh, Jv, h)
    E0 = ctypes.c_double()
    g = ctypes.c_uint64()
    sigma = np.zeros(L * L, dtype=np.int8)
    _check(_load().ttn_oracle_brute_ising(L, _ptr(Jh, ctypes.c_double), _ptr(Jv, ctypes.c_double),
                                          _ptr(h, ctypes.c_double), ctypes.byref(E0),
                                          ctypes.byref(g), _ptr(sigma, ctypes.c_int8)))
    return E0.value, int(g.value), sigma.reshape(L, L)


def brute_potts3(L, Jh, Jv):
    Jh, Jv, _ = _ising_args(L, Jh, Jv, None)
    E0 = ctypes.c_double()
    g = ctypes.c_uint64()
    col = np.zeros(L * L, dtype=np.int8)
    _check(_load().ttn_oracle_brute_potts3(L, _ptr(Jh, ctypes.c_double), _ptr(Jv, ctypes.c_double),
                                           ctypes.byref(E0), ctypes.byref(g),
                                           _ptr(col, ctypes.c_int8)))
    return E0.value, int(g.value), col.reshape(L, L)


def dp_ising(L, Jh, Jv, h=None, count=True, config=False):
    """Site-by-site tropical transfer DP. Returns (E0, g or None, sigma[L,L] or None)."""
    Jh, Jv, h = _ising_args(L, Jh, Jv, h)
    E0 = ctypes.c_double()
    lo = ctypes.c_uint64()
    hi = ctypes.c_uint64()
    sigma = np.zeros(L * L, dtype=np.int8) if config else None
    _check(_load().ttn_oracle_dp_ising(L, _ptr(Jh, ctypes.c_double), _ptr(Jv, ctypes.c_double),
                                       _ptr(h, ctypes.c_double), int(count), int(config),
                                       ctypes.byref(E0), ctypes.byref(lo), ctypes.byref(hi),
                                       _ptr(sigma, ctypes.c_int8)))
    g = (int(hi.value) << 64) | int(lo.value) if count else None
    return E0.value, g, (sigma.reshape(L, L) if config else None)


def dp_potts3(L, Jh, Jv, count=True, config=False):
    Jh, Jv, _ = _ising_args(L, Jh, Jv, None)
    E0 = ctypes.c_double()
    lo = ctypes.c_uint64()
    hi = ctypes.c_uint64()
    col = np.zeros(L * L, dtype=np.int8) if config else None
    _check(_load().ttn_oracle_dp_potts3(L, _ptr(Jh, ctypes.c_double), _ptr(Jv, ctypes.c_double),
                                        int(count), int(config), ctypes.byref(E0),
                                        ctypes.byref(lo), ctypes.byref(hi),
                                        _ptr(col, ctypes.c_int8)))
    g = (int(hi.value) << 64) | int(lo.value) if count else None
    return E0.value, g, (col.reshape(L, L) if config else None)


def ising_energy(L, Jh, Jv, h, sigma) -> float:
    """Eq. (1) PAPER.md:29 evaluated in float64 for a +-1 configuration."""
    Jh, Jv, h = _ising_args(L, Jh, Jv, h)
    s = np.ascontiguousarray(np.asarray(sigma, dtype=np.int8).reshape(-1))
    if s.size != L * L or not np.all(np.abs(s) == 1):
        raise ValueError("sigma must be L*L values of +-1")
    return float(_load().ttn_oracle_ising_energy(L, _ptr(Jh, ctypes.c_double),
                                                 _ptr(Jv, ctypes.c_double),
                                                 _ptr(h, ctypes.c_double),
                                                 _ptr(s, ctypes.c_int8)))


def potts3_energy(L, Jh, Jv, colour) -> float:
    Jh, Jv, _ = _ising_args(L, Jh, Jv, None)
    s = np.ascontiguousarray(np.asarray(colour, dtype=np.int8).reshape(-1))
    return float(_load().ttn_oracle_potts3_energy(L, _ptr(Jh, ctypes.c_double),
                                                  _ptr(Jv, ctypes.c_double),
                                                  _ptr(s, ctypes.c_int8)))
