"""ctypes binding of libising_b200.so — argument marshalling only.

Every function here has the name and meaning of the C entry point in include/ising.h; all
arithmetic of the method runs in the CUDA kernels behind that ABI.  PyTorch supplies device
memory (caching allocator) and the stream through `ising_set_device_hooks`.  There is no
CPU path: importing works without a GPU (so the symbol table can be checked), any compute
call without one raises `IsingError`.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

ISING_LAYOUT_I8 = 0
ISING_LAYOUT_BITS = 1
ISING_RNG_WORDS = 0
ISING_RNG_PLANES = 1
RNG_MODES = {"words": ISING_RNG_WORDS, "planes": ISING_RNG_PLANES}

SYMBOLS = [
    "ising_create", "ising_create_batch", "ising_create_multi", "ising_destroy", "ising_sweep", "ising_sweep_series",
    "ising_observables", "ising_overlap", "ising_overlap_all", "ising_overlap_all_static", "ising_copy_spins", "ising_set_spins", "ising_copy_spins_bits", "ising_set_spins_bits", "ising_set_layout", "ising_set_rng", "ising_set_jit", "ising_last_sweep_specialized",
    "ising_get_counter", "ising_set_counter", "ising_thresholds", "ising_set_device_hooks",
    "ising_synchronize", "ising_kernel_launches", "ising_sweep_path", "ising_force_path",
    "ising_last_error",
]
HEIS_SYMBOLS = [     # include/heisenberg.h
    "heis_create", "heis_destroy", "heis_sweep", "heis_sweep_series", "heis_observables", "heis_copy_spins", "heis_set_spins",
    "heis_get_counter", "heis_set_counter", "heis_sweep_path", "heis_force_generic",
]


class IsingError(RuntimeError):
    pass


_lib = None
_ALLOC_T = C.CFUNCTYPE(C.c_void_p, C.c_size_t)
_FREE_T = C.CFUNCTYPE(None, C.c_void_p)
_live = {}          # device pointer -> torch tensor handed to the library
_hooks = None       # keep the callbacks alive


def lib() -> C.CDLL:
    """Load (building first if stale) the CUDA library; raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path) or _build._stale():
        path = _build.build()
    L = C.CDLL(path)
    vp, i8p, i64p, u64p = C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p
    L.ising_create.restype = vp
    L.ising_create.argtypes = [C.c_int, C.c_int, i8p, C.c_uint64]
    L.ising_create_batch.restype = vp
    L.ising_create_batch.argtypes = [C.c_int, C.c_int, i8p, u64p, C.c_int]
    L.ising_create_multi.restype = vp
    L.ising_create_multi.argtypes = [C.c_int, C.c_int, i8p, u64p, C.c_int, C.c_uint64]
    L.ising_destroy.restype = None
    L.ising_destroy.argtypes = [vp]
    L.ising_sweep.argtypes = [vp, C.c_double, C.c_int, C.c_int, C.c_int]
    L.ising_sweep_series.argtypes = [vp, C.c_double, C.c_int, C.c_int, C.c_int, i64p, i64p]
    L.ising_observables.argtypes = [vp, i64p, i64p]
    L.ising_overlap.argtypes = [vp, C.c_int, C.c_int, i64p]
    L.ising_overlap_all.argtypes = [vp, i64p]
    L.ising_overlap_all_static.argtypes = [i8p, C.c_int, C.c_uint64, i64p, vp]
    L.ising_copy_spins.argtypes = [vp, i8p]
    L.ising_set_spins.argtypes = [vp, i8p]
    L.ising_copy_spins_bits.argtypes = [vp, vp]
    L.ising_set_spins_bits.argtypes = [vp, vp]
    L.ising_set_layout.argtypes = [vp, C.c_int]
    L.ising_set_rng.argtypes = [vp, C.c_int]
    L.ising_set_jit.argtypes = [vp, C.c_int]
    L.ising_last_sweep_specialized.argtypes = [vp]
    L.ising_get_counter.argtypes = [vp, u64p]
    L.ising_set_counter.argtypes = [vp, C.c_uint64]
    L.ising_thresholds.argtypes = [C.c_double, C.c_int, u64p]
    L.ising_set_device_hooks.argtypes = [vp, vp, vp]
    L.ising_synchronize.argtypes = [vp]
    L.ising_kernel_launches.restype = C.c_uint64
    L.ising_sweep_path.restype = C.c_char_p
    L.ising_sweep_path.argtypes = [vp]
    L.ising_force_path.argtypes = [vp, C.c_int]
    L.ising_last_error.restype = C.c_char_p
    L.heis_create.restype = vp
    L.heis_create.argtypes = [C.c_int, C.c_int, C.c_uint64]
    L.heis_destroy.restype = None
    L.heis_destroy.argtypes = [vp]
    L.heis_sweep.argtypes = [vp, C.c_double, C.c_int, C.c_int, C.c_int]
    L.heis_observables.argtypes = [vp, vp, vp]
    L.heis_sweep_series.argtypes = [vp, C.c_double, C.c_int, C.c_int, C.c_int, vp, vp]
    L.heis_copy_spins.argtypes = [vp, vp]
    L.heis_set_spins.argtypes = [vp, vp]
    L.heis_get_counter.argtypes = [vp, u64p]
    L.heis_set_counter.argtypes = [vp, C.c_uint64]
    L.heis_sweep_path.restype = C.c_char_p
    L.heis_sweep_path.argtypes = [vp]
    L.heis_force_generic.argtypes = [vp, C.c_int]
    _lib = L
    return L


def _check(rc: int) -> None:
    if rc != 0:
        raise IsingError(f"libising_b200 error {rc}: {lib().ising_last_error().decode()}")


def use_torch(stream=None) -> None:
    """Route the library's device allocations through torch's caching allocator and its
    launches onto `stream` (default: torch's current stream)."""
    global _hooks
    import torch

    if not torch.cuda.is_available():
        raise IsingError("no CUDA device: libising_b200 has no CPU path")

    def _alloc(n):
        try:
            t = torch.empty(int(n), dtype=torch.uint8, device="cuda")
        except Exception:
            return 0
        _live[t.data_ptr()] = t
        return t.data_ptr()

    def _free(p):
        _live.pop(p, None)

    a, f = _ALLOC_T(_alloc), _FREE_T(_free)
    s = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().ising_set_device_hooks(C.cast(a, C.c_void_p), C.cast(f, C.c_void_p), C.c_void_p(s.cuda_stream)))
    _hooks = (a, f, s)


def _ptr(x):
    """Host numpy array or torch tensor (host or device) -> raw pointer; None -> NULL."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return C.c_void_p(x.ctypes.data)
    return C.c_void_p(x.data_ptr())          # torch tensor


STATIC_MAX_REPLICAS = 64   # ISING_STATIC_MAX_REPLICAS (include/ising.h)


def ising_overlap_all_static(d_spins, n_replicas: int, n_sites: int, d_Q, stream=None) -> None:
    """All pairwise overlaps of n_replicas canonical int8 spin arrays without any device allocation (scratch: a 32 KiB
    __device__ array inside the library, at most STATIC_MAX_REPLICAS replicas).  d_spins, d_Q: DEVICE tensors (int8
    [R*N], int64 [R*R]); stream: a raw cudaStream_t value or None = the library's stream.  Asynchronous; calls that
    overlap on the GPU race on the shared scratch."""
    _check(lib().ising_overlap_all_static(_ptr(d_spins), int(n_replicas), int(n_sites), _ptr(d_Q),
                                          C.c_void_p(int(stream)) if stream else None))


def ising_thresholds(beta: float, dim: int):
    out = np.zeros(3, dtype=np.uint64)
    _check(lib().ising_thresholds(float(beta), int(dim), _ptr(out)))
    return tuple(int(v) for v in out[:dim])


def ising_kernel_launches() -> int:
    return int(lib().ising_kernel_launches())


class Ising:
    """Owner of one `ising_handle`; methods are the C calls of include/ising.h minus the prefix."""

    def __init__(self, dim: int, L: int, coupling=None, seed: int | None = None, seeds=None,
                 rng: str | None = None, sweep_seed: int | None = None):
        if seeds is None:
            seeds = [0 if seed is None else seed]
        sd = np.asarray(list(seeds), dtype=np.uint64)
        self.dim, self.L, self.N, self.R = dim, L, L ** dim, len(sd)
        if coupling is not None and isinstance(coupling, np.ndarray):
            coupling = np.ascontiguousarray(coupling, dtype=np.int8).reshape(-1)
        if sweep_seed is not None:      # ising_create_multi: coupling holds R arrays, sweep randoms shared
            self._h = lib().ising_create_multi(dim, L, _ptr(coupling), _ptr(sd), self.R, int(sweep_seed))
        else:
            self._h = lib().ising_create_batch(dim, L, _ptr(coupling), _ptr(sd), self.R)
        if not self._h:
            raise IsingError(f"ising_create failed: {lib().ising_last_error().decode()}")
        if rng is not None:
            self.set_rng(rng)

    def destroy(self):
        if getattr(self, "_h", None):
            lib().ising_destroy(self._h)
            self._h = None

    __del__ = destroy

    def sweep(self, beta: float, n_sweeps: int, tile: int = 0, k_inner: int = 1) -> None:
        _check(lib().ising_sweep(self._h, float(beta), int(n_sweeps), int(tile), int(k_inner)))

    def sweep_series(self, beta: float, n_sweeps: int, tile: int = 0, k_inner: int = 1, E=None, M=None):
        """E, M: optional caller buffers (numpy or torch int64, n_sweeps*R); default host arrays."""
        if E is None:
            E = np.zeros((n_sweeps, self.R), dtype=np.int64)
        if M is None:
            M = np.zeros((n_sweeps, self.R), dtype=np.int64)
        _check(lib().ising_sweep_series(self._h, float(beta), int(n_sweeps), int(tile), int(k_inner),
                                        _ptr(E), _ptr(M)))
        return E, M

    def observables(self):
        E = np.zeros(self.R, dtype=np.int64)
        M = np.zeros(self.R, dtype=np.int64)
        _check(lib().ising_observables(self._h, _ptr(E), _ptr(M)))
        return E, M

    def overlap(self, a: int, b: int) -> int:
        q = np.zeros(1, dtype=np.int64)
        _check(lib().ising_overlap(self._h, int(a), int(b), _ptr(q)))
        return int(q[0])

    def overlap_all(self, Q=None):
        """(R, R) int64 matrix of all pairwise overlaps; Q: optional caller buffer (numpy or torch, host or device)."""
        if Q is None:
            Q = np.zeros((self.R, self.R), dtype=np.int64)
        _check(lib().ising_overlap_all(self._h, _ptr(Q)))
        return Q

    def copy_spins(self, dst=None):
        if dst is None:
            dst = np.zeros(self.R * self.N, dtype=np.int8)
        _check(lib().ising_copy_spins(self._h, _ptr(dst)))
        return dst

    def set_spins(self, src) -> None:
        if isinstance(src, np.ndarray):
            src = np.ascontiguousarray(src, dtype=np.int8).reshape(-1)
            assert src.size == self.R * self.N
        _check(lib().ising_set_spins(self._h, _ptr(src)))

    def copy_spins_bits(self, dst=None):
        """One bit per site (set = +1): R*N/32 uint32 words; dst numpy or torch (host or device)."""
        if dst is None:
            dst = np.zeros(self.R * self.N // 32, dtype=np.uint32)
        _check(lib().ising_copy_spins_bits(self._h, _ptr(dst)))
        return dst

    def set_spins_bits(self, src) -> None:
        if isinstance(src, np.ndarray):
            src = np.ascontiguousarray(src, dtype=np.uint32).reshape(-1)
            assert src.size == self.R * self.N // 32
        _check(lib().ising_set_spins_bits(self._h, _ptr(src)))

    def set_rng(self, mode) -> None:
        _check(lib().ising_set_rng(self._h, RNG_MODES[mode] if isinstance(mode, str) else int(mode)))

    def set_jit(self, mode) -> None:
        """mode: "auto" (default), "off", "on" or the ISING_JIT_* value."""
        m = {"auto": 0, "off": 1, "on": 2}.get(mode, mode)
        _check(lib().ising_set_jit(self._h, int(m)))

    def last_sweep_specialized(self) -> bool:
        return bool(lib().ising_last_sweep_specialized(self._h))

    def set_layout(self, layout: int) -> None:
        _check(lib().ising_set_layout(self._h, int(layout)))

    @property
    def counter(self) -> int:
        t = np.zeros(1, dtype=np.uint64)
        _check(lib().ising_get_counter(self._h, _ptr(t)))
        return int(t[0])

    @counter.setter
    def counter(self, t: int) -> None:
        _check(lib().ising_set_counter(self._h, int(t)))

    def synchronize(self) -> None:
        _check(lib().ising_synchronize(self._h))

    def sweep_path(self) -> str:
        return lib().ising_sweep_path(self._h).decode()

    def force_path(self, mode) -> None:
        """0 / False: automatic; 1 / True: generic kernels only; 2: a launch per colour (no cluster / grid / data-flow kernel);
        3: no data-flow kernel; 4: no cluster / grid resident kernels (the data-flow kernel may run at any size and k)."""
        _check(lib().ising_force_path(self._h, int(mode)))


class Heisenberg:
    """Owner of one `heis_handle`; methods are the C calls of include/heisenberg.h minus the prefix."""

    def __init__(self, dim: int, L: int, seed: int = 0):
        self.dim, self.L, self.N = dim, L, L ** dim
        self._h = lib().heis_create(dim, L, int(seed))
        if not self._h:
            raise IsingError(f"heis_create failed: {lib().ising_last_error().decode()}")

    def destroy(self):
        if getattr(self, "_h", None):
            lib().heis_destroy(self._h)
            self._h = None

    __del__ = destroy

    def sweep(self, beta: float, n_sweeps: int, tile: int = 0, k_inner: int = 1) -> None:
        _check(lib().heis_sweep(self._h, float(beta), int(n_sweeps), int(tile), int(k_inner)))

    def sweep_series(self, beta: float, n_sweeps: int, tile: int = 0, k_inner: int = 1, E=None, M=None):
        """E (n_sweeps) and M (n_sweeps, 3) after every pass; optional caller buffers (numpy or torch float64)."""
        if E is None:
            E = np.zeros(n_sweeps, dtype=np.float64)
        if M is None:
            M = np.zeros((n_sweeps, 3), dtype=np.float64)
        _check(lib().heis_sweep_series(self._h, float(beta), int(n_sweeps), int(tile), int(k_inner), _ptr(E), _ptr(M)))
        return E, M

    def observables(self):
        E = np.zeros(1, dtype=np.float64)
        M = np.zeros(3, dtype=np.float64)
        _check(lib().heis_observables(self._h, _ptr(E), _ptr(M)))
        return float(E[0]), M

    def copy_spins(self, dst=None):
        """(3, N) float32, component-major; dst may be a numpy array or a torch tensor (host or device)."""
        if dst is None:
            dst = np.zeros((3, self.N), dtype=np.float32)
        _check(lib().heis_copy_spins(self._h, _ptr(dst)))
        return dst

    def set_spins(self, src) -> None:
        if isinstance(src, np.ndarray):
            src = np.ascontiguousarray(src, dtype=np.float32).reshape(-1)
            assert src.size == 3 * self.N
        _check(lib().heis_set_spins(self._h, _ptr(src)))

    @property
    def counter(self) -> int:
        t = np.zeros(1, dtype=np.uint64)
        _check(lib().heis_get_counter(self._h, _ptr(t)))
        return int(t[0])

    @counter.setter
    def counter(self, t: int) -> None:
        _check(lib().heis_set_counter(self._h, int(t)))

    def sweep_path(self) -> str:
        return lib().heis_sweep_path(self._h).decode()

    def force_generic(self, on: bool) -> None:
        _check(lib().heis_force_generic(self._h, int(bool(on))))
