"""Pin of the autocorrelation estimator against a process with a known answer: AR(1), x_t = a x_{t-1} + noise,
has rho(t) = a^t and tau_int = 1/2 + a / (1 - a)."""
import numpy as np

from paper_1006_3865_b200.analysis import autocorrelation, independent_samples_per_second, tau_int


def test_ar1_autocorrelation_time():
    rng = np.random.default_rng(7)
    for a in (0.0, 0.5, 0.9):
        n = 400000
        e = rng.standard_normal(n)
        x = np.empty(n)
        x[0] = e[0]
        for t in range(1, n):
            x[t] = a * x[t - 1] + e[t]
        rho = autocorrelation(x, 5)
        assert abs(rho[1] - a) < 0.01 and abs(rho[2] - a * a) < 0.015
        tau, w = tau_int(x)
        exact = 0.5 + a / (1 - a)
        assert abs(tau - exact) < 0.06 * exact + 0.02, (a, tau, exact)
    assert independent_samples_per_second(1000, 2.0, 5.0) == 50.0
