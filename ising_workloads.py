"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module serves BOTH the CUDA path and the oracle and therefore holds none of the
method's arithmetic (no Metropolis update, no thresholds, no schedule): only the five
workload descriptions of BASELINE.json `configs` and the generator of the quenched ±J
coupling array, which is an *input* of `ising_create` ("harness
couplings").  It imports neither `oracle/` nor `paper_1006_3865_b200/`.

Input recipe: the paper's workloads are hot-start 2D/3D ferromagnets
 and the ±J Edwards–Anderson glass over many realisations; there is no
dataset.  Spins are iid ±1 with p = 1/2 drawn inside `ising_create` from the seed; couplings
are J = +1 (NULL) or iid ±1 with p = 1/2 from `couplings()` below.
"""
from __future__ import annotations

import numpy as np

BETA_C_2D = 0.4406868   # BASELINE.json literal (rounded ln(1+sqrt2)/2)
BETA_C_3D = 0.2216546

# BASELINE.json `configs`, in order.  n = outer passes, tile = T, k = inner sweeps.
CONFIGS = {
    1: dict(dim=2, L=64, seed=1, beta=BETA_C_2D, tile=64, k=1, n=1000),
    2: dict(dim=2, L=1024, seed=2, betas=(0.30, 0.40, BETA_C_2D, 0.50, 0.60), tile=32, k=4, n=10000),
    3: dict(dim=2, L=16384, seed=3, beta=BETA_C_2D, tiles=(32, 64), ks=(1, 4, 16), n=200,
            layouts=("int8", "bits")),
    4: dict(dim=3, L=256, seed=4, beta=BETA_C_3D, tile=8, ks=(1, 4), n=500),
    5: dict(dim=2, L=4096, jseed=5, seeds=tuple(range(100, 116)), beta=1.0, tile=32, k=4, n=1000),
}

_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def _philox4x32_10_np(c0, c1, c2, c3, k0: int, k1: int):
    """Vectorised counter-based generator used ONLY to draw input arrays (uint64 lanes)."""
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        n0 = (p1 >> _S32) ^ c1 ^ np.uint64(k0)
        n1 = p1 & _MASK
        n2 = (p0 >> _S32) ^ c3 ^ np.uint64(k1)
        n3 = p0 & _MASK
        c0, c1, c2, c3 = n0, n1, n2, n3
        k0 = (k0 + _W0) & 0xFFFFFFFF
        k1 = (k1 + _W1) & 0xFFFFFFFF
    return c0, c1, c2, c3


def couplings(dim: int, L: int, jseed: int) -> np.ndarray:
    """Quenched bonds J[d][i] = ±1 (p = 1/2), int8, d-major: bond from site i to i + e_d.

    J[d][i] = -1 if bit 31 of Philox(ctr={i>>2, 2, d, 0}, key=jseed)[i & 3] is set, else +1.
    """
    N = L ** dim
    out = np.empty((dim, N), dtype=np.int8)
    chunk = 1 << 22
    for d in range(dim):
        for g0 in range(0, N // 4 + (1 if N % 4 else 0), chunk):
            g = np.arange(g0, min(g0 + chunk, (N + 3) // 4), dtype=np.uint64)
            z = np.zeros_like(g)
            w = _philox4x32_10_np(g, z + np.uint64(2), z + np.uint64(d), z,
                                  jseed & 0xFFFFFFFF, (jseed >> 32) & 0xFFFFFFFF)
            bits = np.stack([(x >> np.uint64(31)) & np.uint64(1) for x in w], axis=1).reshape(-1)
            lo = 4 * g0
            hi = min(lo + bits.size, N)
            out[d, lo:hi] = 1 - 2 * bits[: hi - lo].astype(np.int8)
    return out.reshape(-1)


def realisations(dim: int, L: int, R: int, jseed: int) -> np.ndarray:
    """R independent +-J coupling arrays (p = 1/2), int8 [R][dim][N], for multi-realisation batches
    (ising_create_multi).  numpy's PCG64 seeded with (jseed, r): fast enough for R = 32 at L = 4096."""
    N = L ** dim
    out = np.empty((R, dim * N), dtype=np.int8)
    for r in range(R):
        bits = np.random.default_rng([jseed, r]).integers(0, 2, size=dim * N, dtype=np.int8)
        out[r] = 1 - 2 * bits
    return out
