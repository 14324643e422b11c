"""ctypes front end of the sequential Heisenberg oracle (oracle/heisenberg_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's CPU legs
import this module.  It never imports paper_1006_3865_b200 and holds no arithmetic of its own.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "heisenberg_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_heisenberg.so")


def build(force: bool = False) -> str:
    """Compile with g++; -ffp-contract=off: every float operation is the one the source states (H1-H8)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u32p, u64p, f32p, f64p = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64), C.POINTER(C.c_float), C.POINTER(C.c_double)
        L.horacle_philox.argtypes = [u32p, u32p, u32p]
        L.horacle_direction.argtypes = [C.c_uint32, C.c_uint32, f32p]
        L.horacle_accept_probability.restype = C.c_float
        L.horacle_accept_probability.argtypes = [C.c_float]
        L.horacle_create.restype = C.c_void_p
        L.horacle_create.argtypes = [C.c_int, C.c_int, C.c_uint64]
        L.horacle_destroy.argtypes = [C.c_void_p]
        L.horacle_sweep.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_int]
        L.horacle_observables.argtypes = [C.c_void_p, f64p, f64p]
        L.horacle_copy_spins.argtypes = [C.c_void_p, f32p]
        L.horacle_set_spins.argtypes = [C.c_void_p, f32p]
        L.horacle_get_counter.restype = C.c_uint64
        L.horacle_get_counter.argtypes = [C.c_void_p]
        L.horacle_set_counter.argtypes = [C.c_void_p, C.c_uint64]
        L.horacle_set_tile_order.argtypes = [C.c_void_p, C.c_int]
        L.horacle_acceptance.argtypes = [C.c_void_p, u64p, u64p]
        _lib = L
    return _lib


def direction(w0: int, w1: int) -> np.ndarray:
    out = np.zeros(3, dtype=np.float32)
    lib().horacle_direction(w0 & 0xFFFFFFFF, w1 & 0xFFFFFFFF, out.ctypes.data_as(C.POINTER(C.c_float)))
    return out


def accept_probability(a: float) -> float:
    return float(lib().horacle_accept_probability(C.c_float(a)))


def philox(ctr, key) -> tuple:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    o = np.zeros(4, dtype=np.uint32)
    p = C.POINTER(C.c_uint32)
    lib().horacle_philox(c.ctypes.data_as(p), k.ctypes.data_as(p), o.ctypes.data_as(p))
    return tuple(int(v) for v in o)


class HeisenbergOracle:
    """Sequential double-checkerboard Metropolis for the O(3) model; spins() is a (3, N) float32 array."""

    def __init__(self, dim: int, L: int, seed: int = 0):
        self._h = lib().horacle_create(dim, L, seed)
        if not self._h:
            raise ValueError(f"bad arguments dim={dim} L={L}")
        self.dim, self.L, self.N = dim, L, L ** dim

    def __del__(self):
        if getattr(self, "_h", None):
            lib().horacle_destroy(self._h)
            self._h = None

    def sweep(self, beta: float, n: int, tile: int = 0, k: int = 1) -> None:
        if lib().horacle_sweep(self._h, beta, n, tile, k) != 0:
            raise ValueError(f"bad sweep arguments beta={beta} n={n} tile={tile} k={k}")

    def observables(self):
        E = C.c_double()
        M = np.zeros(3, dtype=np.float64)
        lib().horacle_observables(self._h, C.byref(E), M.ctypes.data_as(C.POINTER(C.c_double)))
        return E.value, M

    def spins(self) -> np.ndarray:
        out = np.empty((3, self.N), dtype=np.float32)
        lib().horacle_copy_spins(self._h, out.ctypes.data_as(C.POINTER(C.c_float)))
        return out

    def set_spins(self, s) -> None:
        a = np.ascontiguousarray(s, dtype=np.float32).reshape(3, self.N)
        lib().horacle_set_spins(self._h, a.ctypes.data_as(C.POINTER(C.c_float)))

    @property
    def counter(self) -> int:
        return int(lib().horacle_get_counter(self._h))

    @counter.setter
    def counter(self, t: int) -> None:
        lib().horacle_set_counter(self._h, t)

    def set_tile_order(self, reverse: bool) -> None:
        lib().horacle_set_tile_order(self._h, int(reverse))

    def acceptance(self):
        a, n = C.c_uint64(), C.c_uint64()
        lib().horacle_acceptance(self._h, C.byref(a), C.byref(n))
        return a.value, n.value
