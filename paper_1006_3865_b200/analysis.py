"""Time-series helpers for runs of the library (what the multi-hit parameter k costs in
autocorrelation).  Plain numpy on the integer E / M series that `Ising.sweep_series` returns; nothing here
is on the hot path and nothing here touches spins."""
from __future__ import annotations

import numpy as np


def autocorrelation(x, max_lag: int) -> np.ndarray:
    """Normalised autocorrelation rho(0..max_lag) of a 1-D series (FFT, mean removed)."""
    x = np.asarray(x, dtype=np.float64)
    x = x - x.mean()
    n = x.size
    f = np.fft.rfft(x, 2 * n)
    acf = np.fft.irfft(f * np.conj(f))[: max_lag + 1] / np.arange(n, n - max_lag - 1, -1)
    return acf / acf[0] if acf[0] > 0 else np.zeros(max_lag + 1)


def tau_int(x, c: float = 6.0):
    """Integrated autocorrelation time tau = 1/2 + sum_{t>=1} rho(t) with Sokal's automatic window
    (smallest W with W >= c * tau(W)).  Returns (tau, W).  Units: steps of the series."""
    x = np.asarray(x, dtype=np.float64)
    n = x.size
    rho = autocorrelation(x, min(n // 2, 100000))
    tau = 0.5
    for w in range(1, rho.size):
        tau += rho[w]
        if w >= c * tau:
            return float(max(tau, 0.5)), w
    return float(max(tau, 0.5)), rho.size - 1


def independent_samples_per_second(n_steps: int, seconds: float, tau: float) -> float:
    """Effective sample rate: one independent sample per 2 tau steps."""
    return n_steps / (2.0 * tau) / seconds
