"""ctypes front end of the sequential CPU oracle (oracle/ising_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs import this module.  It never imports
paper_1006_3865_b200 and holds no arithmetic of its own — every number comes out of the
C++ file, which cites the passages of the paper (P:n) and of SURVEY.md §8(c) it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ising_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_ising.so")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (plain C++17, libm only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u32p, u64p, i8p, i64p = (C.POINTER(C.c_uint32), C.POINTER(C.c_uint64),
                                 C.POINTER(C.c_int8), C.POINTER(C.c_int64))
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_thresholds.argtypes = [C.c_double, C.c_int, u64p]
        L.oracle_make_couplings.argtypes = [C.c_int, C.c_int, C.c_uint64, i8p]
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [C.c_int, C.c_int, i8p, C.c_uint64]
        L.oracle_create_batch.restype = C.c_void_p
        L.oracle_create_batch.argtypes = [C.c_int, C.c_int, i8p, u64p, C.c_int]
        L.oracle_create_multi.restype = C.c_void_p
        L.oracle_create_multi.argtypes = [C.c_int, C.c_int, i8p, u64p, C.c_int, C.c_uint64]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_sweep.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_int]
        L.oracle_sweep_series.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_int, i64p, i64p]
        L.oracle_observables.argtypes = [C.c_void_p, i64p, i64p]
        L.oracle_overlap.argtypes = [C.c_void_p, C.c_int, C.c_int, i64p]
        L.oracle_copy_spins.argtypes = [C.c_void_p, i8p]
        L.oracle_set_spins.argtypes = [C.c_void_p, i8p]
        L.oracle_get_counter.argtypes = [C.c_void_p, u64p]
        L.oracle_set_counter.argtypes = [C.c_void_p, C.c_uint64]
        L.oracle_set_tile_order.argtypes = [C.c_void_p, C.c_int]
        L.oracle_set_rng.argtypes = [C.c_void_p, C.c_int]
        L.oracle_get_rng.argtypes = [C.c_void_p]
        L.oracle_set_memo.argtypes = [C.c_void_p, C.c_int]
        L.oracle_sweep_random.restype = C.c_uint32
        L.oracle_sweep_random.argtypes = [C.c_void_p, C.c_int, C.c_uint64, C.c_uint64]
        L.oracle_hash.restype = C.c_uint64
        L.oracle_hash.argtypes = [C.c_void_p, C.c_int]
        L.oracle_hash_bytes.restype = C.c_uint64
        L.oracle_hash_bytes.argtypes = [C.c_void_p, C.c_uint64]
        _lib = L
    return _lib


def _p(a: np.ndarray, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def philox4x32_10(ctr, key) -> tuple:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    o = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(o, C.c_uint32))
    return tuple(int(v) for v in o)


def thresholds(beta: float, dim: int) -> tuple:
    o = np.zeros(3, dtype=np.uint64)
    lib().oracle_thresholds(float(beta), int(dim), _p(o, C.c_uint64))
    return tuple(int(v) for v in o[:dim])


def make_couplings(dim: int, L: int, jseed: int) -> np.ndarray:
    out = np.zeros(dim * L ** dim, dtype=np.int8)
    lib().oracle_make_couplings(dim, L, jseed, _p(out, C.c_int8))
    return out


def hash_bytes(a: np.ndarray) -> int:
    a = np.ascontiguousarray(a).view(np.uint8).reshape(-1)
    return int(lib().oracle_hash_bytes(a.ctypes.data, a.size))


RNG_MODES = {"words": 0, "planes": 1}
DEFAULT_RNG = "planes"      # tests flip this to run one body under both mappings


class Oracle:
    """One lattice (or R replicas sharing one coupling array) advanced by the oracle.

    rng: "planes" (default, the product's default mapping) or "words" (SURVEY S8c.3 verbatim)."""

    def __init__(self, dim: int, L: int, seed=None, J: np.ndarray | None = None, seeds=None,
                 rng: str | None = None, sweep_seed: int | None = None):
        if seeds is None:
            seeds = [seed]
        self.dim, self.L, self.N, self.R = dim, L, L ** dim, len(seeds)
        sd = np.asarray(seeds, dtype=np.uint64).copy()
        jp = None
        if J is not None:
            J = np.ascontiguousarray(J, dtype=np.int8).reshape(-1)
            assert J.size == dim * self.N or (sweep_seed is not None and J.size == self.R * dim * self.N)
            jp = _p(J, C.c_int8)
        if sweep_seed is not None:      # multi-realisation batch: J holds R coupling arrays, sweep randoms shared (R17)
            J = np.ascontiguousarray(J, dtype=np.int8).reshape(-1)
            assert J.size == self.R * dim * self.N
            self._h = lib().oracle_create_multi(dim, L, _p(J, C.c_int8), _p(sd, C.c_uint64), self.R, sweep_seed)
        else:
            self._h = lib().oracle_create_batch(dim, L, jp, _p(sd, C.c_uint64), self.R)
        if not self._h:
            raise ValueError("oracle_create_batch rejected its arguments")
        rng = DEFAULT_RNG if rng is None else rng
        self.rng = rng
        if lib().oracle_set_rng(self._h, RNG_MODES[rng]) != 0:
            raise ValueError("bad rng mode")

    def __del__(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    def sweep(self, beta: float, n: int, tile: int = 0, k: int = 1) -> None:
        if lib().oracle_sweep(self._h, beta, n, tile, k) != 0:
            raise ValueError("oracle_sweep rejected its arguments")

    def sweep_series(self, beta: float, n: int, tile: int = 0, k: int = 1):
        E = np.zeros((n, self.R), dtype=np.int64)
        M = np.zeros((n, self.R), dtype=np.int64)
        if lib().oracle_sweep_series(self._h, beta, n, tile, k, _p(E, C.c_int64), _p(M, C.c_int64)) != 0:
            raise ValueError("oracle_sweep_series rejected its arguments")
        return E, M

    def observables(self):
        E = np.zeros(self.R, dtype=np.int64)
        M = np.zeros(self.R, dtype=np.int64)
        lib().oracle_observables(self._h, _p(E, C.c_int64), _p(M, C.c_int64))
        return E, M

    def overlap(self, a: int, b: int) -> int:
        q = C.c_int64(0)
        if lib().oracle_overlap(self._h, a, b, C.byref(q)) != 0:
            raise ValueError("bad replica index")
        return q.value

    def spins(self) -> np.ndarray:
        out = np.zeros(self.R * self.N, dtype=np.int8)
        lib().oracle_copy_spins(self._h, _p(out, C.c_int8))
        return out.reshape(self.R, self.N) if self.R > 1 else out

    def set_spins(self, s: np.ndarray) -> None:
        s = np.ascontiguousarray(s, dtype=np.int8).reshape(-1)
        assert s.size == self.R * self.N
        if lib().oracle_set_spins(self._h, _p(s, C.c_int8)) != 0:
            raise ValueError("spins must be +1/-1")

    @property
    def counter(self) -> int:
        t = C.c_uint64(0)
        lib().oracle_get_counter(self._h, C.byref(t))
        return t.value

    @counter.setter
    def counter(self, t: int) -> None:
        lib().oracle_set_counter(self._h, t)

    def set_memo(self, on: bool) -> None:
        lib().oracle_set_memo(self._h, int(on))

    def sweep_random(self, i: int, H: int, r: int = 0) -> int:
        """The 32-bit random of (replica r, site i, half-sweep H) under this handle's mapping."""
        return int(lib().oracle_sweep_random(self._h, r, i, H))

    def set_tile_order(self, reverse: bool) -> None:
        lib().oracle_set_tile_order(self._h, int(reverse))

    def hash(self, r: int = 0) -> int:
        return int(lib().oracle_hash(self._h, r))
