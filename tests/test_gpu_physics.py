"""High-statistics runs of the CUDA path against exact results.  Parity with the oracle is bit for bit elsewhere; these
runs are too long for the oracle (10^5 .. 10^6 passes) and check what parity cannot: that the random-number mapping and
the schedule give the right physics at a precision of a few 10^-4 (the check the paper itself makes)."""
import math

import numpy as np
import pytest

import ising_workloads as W
from test_oracle_physics import binned, kaufman_u

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1006_3865_b200 as pkg
    pkg.use_torch()
    return pkg


def _energy_series(P, L, seed, beta, tile, k, n, therm, layout="int8", rng="planes"):
    import torch
    g = P.Ising(2, L, seed=seed, rng=rng)
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(beta, therm, tile, k)
    E = torch.zeros(n, dtype=torch.int64, device="cuda")
    M = torch.zeros(n, dtype=torch.int64, device="cuda")
    g.sweep_series(beta, n, tile, k, E=E, M=M)
    return E.cpu().numpy().astype(np.float64), M.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("L,tile,k,layout,rng,n", [
    (64, 32, 1, "int8", "planes", 1000000),
    (64, 32, 4, "bits", "planes", 300000),       # multi-hit: a different chain, the same equilibrium
    (128, 64, 1, "int8", "planes", 300000),
    (64, 32, 1, "int8", "words", 300000),
    (64, 64, 1, "int8", "planes", 300000),       # plain checkerboard (config 1 shape)
    (128, 128, 1, "int8", "planes", 200000),     # plain checkerboard on the cluster-resident kernel
    (128, 16, 1, "int8", "planes", 200000),      # the paper's tile size: masked half-sweeps
])
def test_energy_at_the_critical_point_matches_kaufman(P, L, tile, k, layout, rng, n):
    """<E>/N at beta_c on the periodic L x L lattice against Kaufman's exact finite-lattice value."""
    u = kaufman_u(L, W.BETA_C_2D)
    E, _ = _energy_series(P, L, 100 + L + k, W.BETA_C_2D, tile, k, n, 5000, layout, rng)
    mean, err = binned(E / (L * L), nbins=50)
    assert abs(mean - u) < 4 * err, (mean, u, err)
    assert err < 2.5e-3, err          # critical slowing down: tau_int of E is about 50 passes at L = 64, more at 128


def test_magnetisation_below_tc_matches_yang(P):
    """|M|/N at beta = 0.6 from a cold start against Yang's spontaneous magnetisation (finite-size correction at
    L = 256 is far below the error bar)."""
    import torch
    beta, L = 0.6, 256
    m0 = (1 - math.sinh(2 * beta) ** -4) ** 0.125
    g = P.Ising(2, L, seed=77)
    g.set_spins(np.ones(L * L, dtype=np.int8))
    g.sweep(beta, 2000, 32, 1)
    M = torch.zeros(40000, dtype=torch.int64, device="cuda")
    E = torch.zeros(40000, dtype=torch.int64, device="cuda")
    g.sweep_series(beta, 40000, 32, 1, E=E, M=M)
    mean, err = binned(np.abs(M.cpu().numpy().astype(np.float64)) / (L * L), nbins=40)
    assert abs(mean - m0) < max(4 * err, 2e-4), (mean, m0, err)
    assert err < 2e-4


def test_resident_kernel_equilibrium(P):
    """The cluster-resident kernel over 2 x 10^5 passes in blocks of 50 (one launch each): energy at beta_c, L = 128."""
    L, T = 128, 32
    u = kaufman_u(L, W.BETA_C_2D)
    g = P.Ising(2, L, seed=5)
    g.sweep(W.BETA_C_2D, 5000, T, 1)
    assert g.sweep_path() == "resident_planes_i8"
    Es = []
    for _ in range(4000):
        g.sweep(W.BETA_C_2D, 50, T, 1)
        Es.append(int(g.observables()[0][0]))
    mean, err = binned(np.asarray(Es, dtype=np.float64) / (L * L), nbins=40)
    assert abs(mean - u) < 4 * err, (mean, u, err)
    assert err < 3e-3


def test_heisenberg_high_temperature_series_3d(P):
    """Heisenberg 3D L = 16, beta = 0.2, tile 8: bond correlation against L(K) + 4 L(K)^3 (+ O(K^5) ~ 1e-4)."""
    beta, L = 0.2, 16
    g = P.Heisenberg(3, L, seed=9)
    g.sweep(beta, 500, 8, 1)
    assert g.sweep_path() == "heis_tile"
    Es, _ = g.sweep_series(beta, 12000, 8, 1)
    nb = 3 * L ** 3
    mean, err = binned(np.asarray(Es) / nb, nbins=40)
    lang = 1 / math.tanh(beta) - 1 / beta
    assert abs(mean + (lang + 4 * lang ** 3)) < 4 * err + 2e-4, (mean, lang + 4 * lang ** 3, err)
    assert err < 1e-4


def test_3d_equilibrium_is_the_same_for_both_schedules(P):
    """3D Ising L = 16 at the critical coupling: the double checkerboard with 8^3 tiles (cluster-resident kernel, E counted
    on the registers) and the plain checkerboard (tile = L, the same kernel in plain mode) are different chains with the same
    equilibrium; no exact finite-lattice value exists in 3D, so the two are compared with each other."""
    import torch
    L, beta = 16, W.BETA_C_3D
    means = []
    for tile, k, n, path in ((8, 1, 200000, "resident3d_planes_i8"), (8, 2, 100000, "resident3d_planes_i8"), (16, 1, 100000, "resident3d_plain_i8")):
        g = P.Ising(3, L, seed=31 + tile + k)
        g.sweep(beta, 3000, tile, k)
        E = torch.zeros(n, dtype=torch.int64, device="cuda")
        M = torch.zeros(n, dtype=torch.int64, device="cuda")
        g.sweep_series(beta, n, tile, k, E=E, M=M)
        assert g.sweep_path() == path
        means.append(binned(E.cpu().numpy().astype(np.float64) / L ** 3, nbins=40))
    (m0, e0), (m1, e1), (m2, e2) = means
    assert abs(m0 - m2) < 4 * math.hypot(e0, e2), means
    assert abs(m1 - m2) < 4 * math.hypot(e1, e2), means
    assert max(e0, e1, e2) < 4e-3 and -1.1 < m0 < -0.9          # u_c = -0.99 in the infinite lattice
