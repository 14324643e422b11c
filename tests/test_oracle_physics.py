"""Physics pins of the oracle: exact enumeration, Kaufman / Onsager / Yang closed forms,
detailed balance.  All independent of oracle/ (numpy + mpmath restate the *definitions*,
the oracle runs the *algorithm*).  BASELINE.json north_star, "validated three ways".

Statistical checks use fixed seeds, so they are deterministic; the bar is the 3σ of
north_star with σ from a binning analysis of the oracle's own time series.
"""
import itertools
import math

import numpy as np
import pytest

pytestmark = pytest.mark.usefixtures("both_rngs")

BETA_C = 0.4406868


# ------------------------------------------------------------------ helpers (definitions only)
def enumerate_2d(L):
    """All 2^(L*L) states of the periodic L×L lattice: E = -Σ s_i (s_right + s_down), M = Σ s."""
    n = L * L
    idx = np.arange(2 ** n, dtype=np.int64)
    s = 1 - 2 * ((idx[:, None] >> np.arange(n)) & 1).astype(np.int8)  # bit i ↔ site i = x + L*y
    s = s.reshape(-1, L, L)  # [state, y, x]
    E = -(s * np.roll(s, -1, axis=2)).sum(axis=(1, 2), dtype=np.int64) \
        - (s * np.roll(s, -1, axis=1)).sum(axis=(1, 2), dtype=np.int64)
    M = s.sum(axis=(1, 2), dtype=np.int64)
    return s.reshape(-1, n), E, M


def enumerate_3d_L2():
    n = 8
    idx = np.arange(2 ** n, dtype=np.int64)
    s = 1 - 2 * ((idx[:, None] >> np.arange(n)) & 1).astype(np.int8)
    s3 = s.reshape(-1, 2, 2, 2)  # [state, z, y, x]
    E = np.zeros(2 ** n, dtype=np.int64)
    for ax in (1, 2, 3):  # each site owns its +e_d bond; for L = 2 every pair carries two bonds
        E -= (s3 * np.roll(s3, -1, axis=ax)).sum(axis=(1, 2, 3), dtype=np.int64)
    return s, E, s.sum(axis=1, dtype=np.int64)


def boltzmann_mean(E, beta, obs):
    w = np.exp(-beta * (E - E.min()))
    return float((w * obs).sum() / w.sum())


def binned(series, nbins=40):
    x = np.asarray(series, dtype=np.float64)
    nb = len(x) // nbins
    b = x[: nb * nbins].reshape(nbins, nb).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nbins)


def mc_series(orc, dim, L, seed, beta, tile, k, n, therm=2000):
    o = orc.Oracle(dim, L, seed=seed)
    o.sweep(beta, therm, tile, k)
    E, M = o.sweep_series(beta, n, tile, k)
    return E[:, 0], M[:, 0]


def kaufman_lnZ(L, beta):
    """ln Z of the periodic L×L Ising model (Kaufman 1949), J = 1, in mpmath."""
    import mpmath as mp
    K = mp.mpf(beta)
    N = L * L

    def gamma(l):
        if l == 0:
            return 2 * K + mp.log(mp.tanh(K))
        return mp.acosh(mp.cosh(2 * K) ** 2 / mp.sinh(2 * K) - mp.cos(mp.pi * l / L))

    p = [mp.mpf(1)] * 4
    for r in range(L):
        go, ge = gamma(2 * r + 1), gamma(2 * r)
        p[0] *= 2 * mp.cosh(L * go / 2)
        p[1] *= 2 * mp.sinh(L * go / 2)
        p[2] *= 2 * mp.cosh(L * ge / 2)
        p[3] *= 2 * mp.sinh(L * ge / 2)
    return mp.log(mp.mpf(1) / 2) + (mp.mpf(N) / 2) * mp.log(2 * mp.sinh(2 * K)) + mp.log(sum(p))


def kaufman_u(L, beta):
    import mpmath as mp
    mp.mp.dps = 40
    return float(-mp.diff(lambda b: kaufman_lnZ(L, b), mp.mpf(beta)) / (L * L))


# ------------------------------------------------------------------ the pins
def test_definitions_reproduce_survey_numbers():
    """Sanity of the test's own restatements: brute force 4×4 and Kaufman agree with each
    other and with the values printed in SURVEY.md §8(c) 'Pins'."""
    import mpmath as mp
    mp.mp.dps = 40
    _, E, M = enumerate_2d(4)
    assert boltzmann_mean(E, BETA_C, E) == pytest.approx(-25.049981021, abs=1e-8)
    assert boltzmann_mean(E, BETA_C, np.abs(M)) == pytest.approx(13.5017672896, abs=1e-8)
    lnZ_bf = math.log(np.exp(-BETA_C * (E - E.min())).sum()) - BETA_C * E.min()
    assert float(kaufman_lnZ(4, BETA_C)) == pytest.approx(lnZ_bf, rel=1e-12)
    assert kaufman_u(4, BETA_C) == pytest.approx(-25.049981021 / 16, abs=1e-9)
    assert kaufman_u(16, BETA_C) == pytest.approx(-1.4530649029, abs=1e-9)
    assert kaufman_u(16, 0.30) == pytest.approx(-0.704532670859, abs=1e-9)
    assert kaufman_u(64, BETA_C) == pytest.approx(-1.4239384631, abs=1e-8)


@pytest.mark.parametrize("tile,k,seed", [(4, 1, 11), (2, 1, 12), (2, 4, 13)])
@pytest.mark.parametrize("beta", [0.30, BETA_C, 0.60])
def test_exact_enumeration_4x4(orc, tile, k, seed, beta):
    """MC ⟨E⟩, ⟨|M|⟩, ⟨E²⟩ on the 4×4 lattice within 3σ of the 2^16-state sums (north_star):
    a biased acceptance rule, a wrong threshold index or a correlated RNG→site map fails."""
    _, Ee, Me = enumerate_2d(4)
    E, M = mc_series(orc, 2, 4, seed, beta, tile, k, 400000)
    for name, obs_mc, obs_ex in [("E", E, Ee), ("|M|", np.abs(M), np.abs(Me)), ("E2", E.astype(float) ** 2, Ee.astype(float) ** 2)]:
        mean, err = binned(obs_mc)
        exact = boltzmann_mean(Ee, beta, obs_ex)
        assert abs(mean - exact) < 3 * err, (name, mean, exact, err)
        assert err < 0.01 * max(1.0, abs(exact))  # the test has resolving power


def test_exact_enumeration_2x2x2(orc):
    """3D path on the smallest lattice (256 states, doubled bonds), β = 0.2216546."""
    beta = 0.2216546
    _, Ee, Me = enumerate_3d_L2()
    assert boltzmann_mean(Ee, beta, Ee) == pytest.approx(-14.0102333, abs=1e-6)
    assert boltzmann_mean(Ee, beta, np.abs(Me)) == pytest.approx(5.49671243, abs=1e-7)
    E, M = mc_series(orc, 3, 2, 21, beta, 2, 1, 600000)
    for obs_mc, obs_ex in [(E, Ee), (np.abs(M), np.abs(Me))]:
        mean, err = binned(obs_mc)
        assert abs(mean - boltzmann_mean(Ee, beta, obs_ex)) < 3 * err


def test_single_site_detailed_balance_2x2(orc):
    """π(a) P(a→b) = π(b) P(b→a) for all 16 states × 4 sites of the 2×2 lattice, with the
    oracle's integer thresholds as P: violated by less than 2^-32 · π (SURVEY §8(c) '2×2' (i))."""
    s, E, _ = enumerate_2d(2)
    for beta in (0.2, BETA_C, 1.0):
        thr = orc.thresholds(beta, 2)

        def P(dE):
            return 1.0 if dE <= 0 else thr[dE // 4 - 1] / 2.0 ** 32

        for a in range(16):
            for site in range(4):
                b = a ^ (1 << site)
                dE = int(E[b] - E[a])
                assert dE % 4 == 0 and abs(dE) <= 8
                lhs = math.exp(-beta * E[a]) * P(dE)
                rhs = math.exp(-beta * E[b]) * P(-dE)
                # P is the exact probability rounded down by < 2^-32 (absolute)
                worst = max(math.exp(-beta * E[a]), math.exp(-beta * E[b]))
                assert abs(lhs - rhs) <= 2.0 ** -32 * worst * (1 + 1e-9)


def test_visit_histogram_2x2(orc):
    """χ² of the visited-state histogram against Boltzmann weights restricted to the 12-state
    class of the start (the 2×2 chain is reducible: SURVEY §8(c) '2×2' (ii))."""
    s, E, M = enumerate_2d(2)
    # the closed 4-cycle: both sub-lattices anti-aligned (E = 0, M = 0, s0 = -s3, s1 = -s2)
    cyc = [a for a in range(16) if s[a][0] == -s[a][3] and s[a][1] == -s[a][2]]
    assert len(cyc) == 4 and all(E[a] == 0 and M[a] == 0 for a in cyc)
    allowed = [a for a in range(16) if a not in cyc]
    beta = BETA_C
    w = np.exp(-beta * E[allowed].astype(float))
    w /= w.sum()
    assert (w * E[allowed]).sum() == pytest.approx(-7.1455001, abs=1e-6)  # SURVEY value
    o = None
    for seed in range(31, 40):
        o = orc.Oracle(2, 2, seed=seed)
        code = int(((1 - o.spins().astype(np.int64)) // 2 * (1 << np.arange(4))).sum())
        if code in allowed:
            break
    counts = np.zeros(16, dtype=np.int64)
    n, thin = 60000, 3
    for _ in range(n):
        o.sweep(beta, thin, 2, 1)
        code = int(((1 - o.spins().astype(np.int64)) // 2 * (1 << np.arange(4))).sum())
        counts[code] += 1
    assert counts[cyc].sum() == 0
    exp = w * n
    chi2 = float(((counts[allowed] - exp) ** 2 / exp).sum())
    assert chi2 < 35.0, chi2   # 11 dof: p(χ² > 35) ≈ 2.5e-4 (thinned, so nearly independent)
    emean = (counts[allowed] * E[allowed]).sum() / n
    assert emean == pytest.approx(-7.1455001, abs=0.03)
    assert abs(emean - (-6.7882251)) > 0.2   # and NOT the full 16-state value


@pytest.mark.parametrize("beta,tile,k,seed", [(0.30, 4, 2, 41), (BETA_C, 16, 1, 42), (BETA_C, 8, 1, 44), (0.60, 8, 4, 43)])
def test_kaufman_energy_L16(orc, beta, tile, k, seed):
    """⟨E⟩/N at L = 16 against Kaufman's exact finite-lattice result (the check the paper
    itself uses, P:84 / ref. [20]); at β_c this is the finite-size companion of u → -√2."""
    u = kaufman_u(16, beta)
    E, _ = mc_series(orc, 2, 16, seed, beta, tile, k, 60000, therm=3000)
    mean, err = binned(E / 256.0)
    assert abs(mean - u) < 3 * err, (mean, u, err)
    assert err < 0.004


def test_onsager_limit_and_yang_magnetisation(orc):
    """u(β_c) → -√2 as L grows (north_star) and Yang's m0 below T_c from a cold start."""
    assert kaufman_u(256, 0.44068679350977147) == pytest.approx(-math.sqrt(2), abs=0.01)
    beta = 0.6
    m0 = (1 - math.sinh(2 * beta) ** -4) ** 0.125
    assert m0 == pytest.approx(0.973608667, abs=1e-8)
    o = orc.Oracle(2, 64, seed=51)
    o.set_spins(np.ones(64 * 64, dtype=np.int8))
    o.sweep(beta, 300, 32, 1)
    _, M = o.sweep_series(beta, 3000, 32, 1)
    mean, err = binned(np.abs(M[:, 0]) / 4096.0, nbins=20)
    assert abs(mean - m0) < max(3 * err, 1e-3), (mean, m0, err)
