"""Pins of the Heisenberg oracle (oracle/heisenberg_oracle.cpp, readings H1-H8) against what the mathematics
fixes: closed forms, exact finite-system results, series, invariants.  CPU only."""
import math

import numpy as np
import pytest

from oracle import heisenberg as H


# ---- H2: the direction map against its closed form in double precision -------------------------------
def closed_form_direction(wa, wb):
    z = (wa >> 12) * 2.0 ** -19 - 1.0
    phi20 = ((wa & 0xFFF) << 8) | (wb >> 24)
    phi = phi20 * 2.0 ** -17 * (math.pi / 4)          # octant + fraction, in units of pi/4
    rho = math.sqrt(max(0.0, 1.0 - z * z))
    return np.array([rho * math.cos(phi), rho * math.sin(phi), z])


def test_direction_matches_closed_form():
    rs = np.random.RandomState(1)
    words = [(int(a), int(b)) for a, b in rs.randint(0, 2 ** 32, size=(20000, 2), dtype=np.uint64)]
    # octant boundaries and extreme heights
    for q in range(8):
        for frac in (0, 1, 0x1FFFF, 0x10000):
            phi20 = (q << 17) | frac
            words.append((0x80000000 | (phi20 >> 8), (phi20 & 0xFF) << 24))
    words += [(0, 0), (0xFFFFFFFF, 0xFFFFFFFF), (0xFFF, 0xFF000000), (0x1000, 0x00FFFFFF)]
    worst = 0.0
    for w0, w1 in words:
        d = H.direction(w0, w1).astype(np.float64)
        worst = max(worst, float(np.max(np.abs(d - closed_form_direction(w0, w1)))))
        assert abs(float(np.dot(d, d)) - 1.0) < 6e-7
    assert worst < 2.5e-7, worst      # a few float ulps; a wrong quadrant, sign or coefficient is >= 1e-4


def test_direction_is_a_pure_function_of_the_stated_bits():
    # H2 uses all of wa and bits 31..24 of wb only (the low 24 bits of wb are the acceptance number)
    a = H.direction(0x12345678, 0x89ABCDEF)
    assert np.array_equal(a, H.direction(0x12345678, 0x89000000))
    assert not np.array_equal(a, H.direction(0x12345679, 0x89ABCDEF))
    assert not np.array_equal(a, H.direction(0x12345678, 0x8AABCDEF))
    assert not np.array_equal(a, H.direction(0x12346678, 0x89ABCDEF))


# ---- H6: the acceptance probability against exp ---------------------------------------------------
def test_accept_probability_matches_exp():
    worst = 0.0
    for a in np.concatenate([-np.logspace(-6, math.log10(44.0), 4000), -np.linspace(0.0, 44.0, 3001)[1:]]):
        af = float(np.float32(a))
        p = H.accept_probability(af)
        worst = max(worst, abs(p / math.exp(af) - 1.0))
    assert worst < 4e-6, worst
    assert H.accept_probability(-44.5) == 0.0 and H.accept_probability(-1e30) == 0.0   # tt < -64: never (H6)
    assert 0.0 < H.accept_probability(-44.0) < 1e-19
    assert H.accept_probability(-1e-30) == 1.0


def test_accept_probability_is_monotone_on_a_fine_grid():
    a = np.float32(-3.0)
    prev = H.accept_probability(float(a))
    for _ in range(20000):                       # consecutive floats across several n = rint(tt) boundaries
        a = np.nextafter(a, np.float32(0.0))
        p = H.accept_probability(float(a))
        assert p >= prev * (1.0 - 3e-7)
        prev = p


# ---- H3: hot start = uniform on the sphere --------------------------------------------------------
def test_hot_start_moments_of_the_uniform_sphere():
    o = H.HeisenbergOracle(2, 512, seed=11)
    s = o.spins().astype(np.float64)
    n = s.shape[1]
    assert np.max(np.abs(np.sum(s * s, axis=0) - 1.0)) < 6e-7
    sig = 4.5 / math.sqrt(n)
    for c in range(3):
        assert abs(s[c].mean()) < sig * math.sqrt(1 / 3)                       # <s_c> = 0, var 1/3
        assert abs((s[c] ** 2).mean() - 1 / 3) < sig * math.sqrt(1 / 5 - 1 / 9)   # <s_c^2> = 1/3, <s_c^4> = 1/5
        assert abs((s[c] ** 4).mean() - 1 / 5) < sig * math.sqrt(1 / 9 - 1 / 25)  # <s_c^8> = 1/9
    for a, b in ((0, 1), (0, 2), (1, 2)):
        assert abs((s[a] * s[b]).mean()) < sig * math.sqrt(1 / 15)             # <s_a^2 s_b^2> = 1/15
    # the first site follows H3 literally
    w = H.philox([0, 6, 0, 0], [11, 0])
    assert np.array_equal(o.spins()[:, 0], H.direction(w[0], w[1]))
    assert np.array_equal(o.spins()[:, 1], H.direction(w[2], w[3]))
    w = H.philox([77 >> 1, 6, 0, 0], [11, 0])
    assert np.array_equal(o.spins()[:, 77], H.direction(w[2], w[3]))


# ---- H8: energy of spin spirals (closed form), pins the neighbour indexing of E in 1D/2D/3D ----------
@pytest.mark.parametrize("dim,L,n", [(1, 12, (5,)), (2, 8, (1, 3)), (3, 6, (1, 2, 0)), (3, 4, (0, 1, 3))])
def test_energy_of_a_spin_spiral(dim, L, n):
    o = H.HeisenbergOracle(dim, L, seed=0)
    idx = np.arange(L ** dim)
    xyz = [(idx // L ** d) % L for d in range(dim)]
    q = [2 * math.pi * nd / L for nd in n]
    phase = sum(qd * xd for qd, xd in zip(q, xyz))
    s = np.stack([np.cos(phase), np.sin(phase), np.zeros_like(phase)]).astype(np.float32)
    o.set_spins(s)
    E, M = o.observables()
    assert abs(E - (-(L ** dim) * sum(math.cos(qd) for qd in q))) < 1e-4 * L ** dim
    assert np.all(np.abs(M) < 1e-3)


def test_energy_and_magnetisation_of_the_aligned_state():
    for dim, L in ((1, 6), (2, 6), (3, 4), (2, 2), (3, 2)):
        o = H.HeisenbergOracle(dim, L, seed=0)
        s = np.zeros((3, L ** dim), dtype=np.float32)
        s[1] = 1.0
        o.set_spins(s)
        E, M = o.observables()
        assert E == -dim * L ** dim and tuple(M) == (0.0, float(L ** dim), 0.0)


# ---- H5: the local field against E: with P = 0 (huge beta) only moves with dE <= 0 pass, so the energy H8
# (pinned above independently) can never rise.  A wrong neighbour, sign or component in the field breaks it.
@pytest.mark.parametrize("dim,L,T", [(1, 16, 4), (2, 8, 4), (2, 8, 8), (3, 4, 2), (3, 4, 4)])
def test_quench_energy_is_monotone(dim, L, T):
    o = H.HeisenbergOracle(dim, L, seed=5)
    E_prev, _ = o.observables()
    for _ in range(40):
        o.sweep(1e6, 1, T, 1)
        E, _ = o.observables()
        assert E <= E_prev + 1e-4
        E_prev = E
    assert E_prev < -0.7 * dim * L ** dim          # and it does go down, towards -dim*N
    s = o.spins().astype(np.float64)
    assert np.max(np.abs(np.sum(s * s, axis=0) - 1.0)) < 6e-7


def test_beta_zero_accepts_everything():
    o = H.HeisenbergOracle(2, 8, seed=3)
    o.sweep(0.0, 3, 4, 2)
    a, n = o.acceptance()
    assert a == n == 3 * 2 * 64
    # and the last proposal of site 0 (colour 0, inner sweep t = 5, H = 10) is what H4/H2 say
    w = H.philox([0, 5, 10, 0], [3, 0])
    assert np.array_equal(o.spins()[:, 0], H.direction(w[0], w[1]))
    assert np.array_equal(o.spins()[:, 8 + 1], H.direction(w[2], w[3]))     # (1, 1): same block, row 1, colour 0
    w = H.philox([0, 5, 11, 0], [3, 0])            # colour 1, H = 11: sites (1, 0) and (0, 1) of block 0
    assert np.array_equal(o.spins()[:, 1], H.direction(w[0], w[1]))
    assert np.array_equal(o.spins()[:, 8], H.direction(w[2], w[3]))
    w = H.philox([(5 >> 1) * 4 + (6 >> 1), 5, 10, 0], [3, 0])              # site (6, 4): block row 2, block column 3
    assert np.array_equal(o.spins()[:, 4 * 8 + 6], H.direction(w[0], w[1]))


# ---- exact finite systems: Joyce (1967), ring of N classical Heisenberg spins -------------------------
def ring_energy(N, K):
    """<sum over the N bonds of s_i.s_(i+1)> for the closed ring: Z_N = sum_l (2l+1) i_l(K)^N."""
    from scipy.special import spherical_in
    ls = np.arange(0, 60)
    il = spherical_in(ls, K)
    dil = spherical_in(ls, K, derivative=True)
    Z = np.sum((2 * ls + 1) * il ** N)
    dZ = np.sum((2 * ls + 1) * N * il ** (N - 1) * dil)
    return dZ / Z


def mean_energy(o, beta, T, sweeps, therm, block=500):
    o.sweep(beta, therm, T, 1)
    Es = np.empty(sweeps)
    for i in range(sweeps):
        o.sweep(beta, 1, T, 1)
        Es[i] = o.observables()[0]
    b = Es[: sweeps // block * block].reshape(-1, block).mean(axis=1)
    return Es.mean(), b.std(ddof=1) / math.sqrt(len(b))


def test_ring_energy_closed_form_reduces_to_langevin():
    # sanity of the formula itself: for a long ring the bond correlation is the Langevin function coth K - 1/K
    K = 1.3
    assert abs(ring_energy(400, K) / 400 - (1 / math.tanh(K) - 1 / K)) < 1e-12


@pytest.mark.parametrize("beta", [0.7, 2.0])
def test_ring_of_eight_matches_joyce(beta):
    o = H.HeisenbergOracle(1, 8, seed=21)
    E, err = mean_energy(o, beta, 4, 200000, 2000)
    exact = -ring_energy(8, beta)
    assert abs(E - exact) < 4.5 * err + 1e-3, (E, exact, err)
    assert err < 0.02


def test_two_by_two_torus_is_a_ring_of_four_with_double_bonds():
    beta = 0.6
    o = H.HeisenbergOracle(2, 2, seed=22)
    E, err = mean_energy(o, beta, 2, 200000, 2000)
    exact = -2.0 * ring_energy(4, 2.0 * beta)
    assert abs(E - exact) < 4.5 * err + 1e-3, (E, exact, err)


def test_high_temperature_series_3d():
    # bond correlation <s_i.s_j> = L(K) + 2(d-1) L(K)^3 + O(K^5) on the hypercubic lattice (L >= 6: no wrapping 3-paths)
    beta, L = 0.2, 6
    o = H.HeisenbergOracle(3, L, seed=23)
    E, err = mean_energy(o, beta, 6, 6000, 200, block=200)
    lang = 1 / math.tanh(beta) - 1 / beta
    series = -(3 * L ** 3) * (lang + 4 * lang ** 3)
    assert abs(E - series) / (3 * L ** 3) < 4.5 * err / (3 * L ** 3) + 2e-4, (E, series, err)


# ---- H7: schedule invariants -------------------------------------------------------------------------
@pytest.mark.parametrize("dim,L,T", [(2, 16, 4), (3, 8, 4), (1, 16, 4)])
def test_sweeps_compose_and_tile_order_is_irrelevant(dim, L, T):
    a, b, c = (H.HeisenbergOracle(dim, L, seed=9) for _ in range(3))
    a.sweep(0.8, 5, T, 2)
    b.sweep(0.8, 2, T, 2); b.sweep(0.8, 3, T, 2)
    c.set_tile_order(True); c.sweep(0.8, 5, T, 2)
    assert a.counter == b.counter == 10
    assert np.array_equal(a.spins(), b.spins()) and np.array_equal(a.spins(), c.spins())
    d = H.HeisenbergOracle(dim, L, seed=9)
    d.sweep(0.8, 5, L, 2)                      # plain checkerboard: a different (valid) trajectory (S8c reading 5)
    assert not np.array_equal(a.spins(), d.spins())
    e = H.HeisenbergOracle(dim, L, seed=10)
    e.sweep(0.8, 5, T, 2)
    assert not np.array_equal(a.spins(), e.spins())


def test_argument_checks():
    with pytest.raises(ValueError):
        H.HeisenbergOracle(2, 7)
    with pytest.raises(ValueError):
        H.HeisenbergOracle(4, 8)
    o = H.HeisenbergOracle(2, 12, seed=1)
    for bad in ((0.5, 1, 5, 1), (0.5, 1, 4, 1), (0.5, 1, 6, 0), (-1.0, 1, 6, 1), (0.5, -1, 6, 1)):
        with pytest.raises(ValueError):
            o.sweep(*bad)          # T=5 odd; T=4 -> B=3 odd; k=0; beta<0; n<0
