"""Exact (bitwise) invariants of the oracle — SURVEY.md §8(c) "Exact invariants".

Each one is a property the mathematics fixes, so a slip in the corresponding part of the
oracle (a neighbour index, the back-bond J_d(i-e_d), the multi-hit counter, the colour
rule) breaks it.
"""
import numpy as np
import pytest

import ising_workloads as W

pytestmark = pytest.mark.usefixtures("both_rngs")

BETA_C = 0.4406868


def state(o, r=0):
    E, M = o.observables()
    return int(E[r]), int(M[r]), o.hash(r)


@pytest.mark.parametrize("dim,L", [(2, 2), (2, 4), (2, 16), (3, 2), (3, 4), (3, 8)])
def test_ground_state_energy(orc, dim, L):
    """E(all +1) = -dim·N for J = +1 (north_star: -2N in 2D, -3N in 3D); M = N."""
    o = orc.Oracle(dim, L, seed=1)
    o.set_spins(np.ones(L ** dim, dtype=np.int8))
    E, M = o.observables()
    assert (int(E[0]), int(M[0])) == (-dim * L ** dim, L ** dim)
    # β = 40: every proposed flip costs ΔE > 0 and thr = 0 ⇒ nothing moves
    o.sweep(40.0, 3, 2, 2)
    assert state(o)[:2] == (-dim * L ** dim, L ** dim)


def test_energy_definition_against_numpy(orc):
    """E and M of a random state vs the definition written with numpy rolls (2D, 3D, ±J)."""
    for dim, L in [(2, 12), (3, 6)]:
        J = W.couplings(dim, L, 9)
        o = orc.Oracle(dim, L, seed=5, J=J)
        s = o.spins().astype(np.int64).reshape((L,) * dim)          # [z,]y,x
        Jd = J.astype(np.int64).reshape((dim,) + (L,) * dim)
        E = 0
        for d in range(dim):
            ax = dim - 1 - d                                       # e_0 = x is the last axis
            E -= int((Jd[d] * s * np.roll(s, -1, axis=ax)).sum())
        assert state(o)[:2] == (E, int(s.sum()))


def test_parity_of_E_and_M(orc):
    """Every flip changes E by a multiple of 4 and M by 2."""
    o = orc.Oracle(2, 16, seed=3)
    E0, M0, _ = state(o)
    E, M = o.sweep_series(BETA_C, 50, 4, 2)
    assert np.all((E[:, 0] - E0) % 4 == 0) and np.all((M[:, 0] - M0) % 2 == 0)
    assert np.all((E[:, 0] + 2 * 256) % 4 == 0)   # E ≡ -dim·N (mod 4) for J = +1


@pytest.mark.parametrize("dim,L,tile,k", [(2, 16, 4, 3), (2, 16, 16, 1), (3, 8, 4, 2)])
def test_sweep_is_additive_and_reproducible(orc, dim, L, tile, k):
    """sweep(a); sweep(b) ≡ sweep(a+b); same seed ⇒ same bits; the counter advances by n·k."""
    beta = 0.3
    a = orc.Oracle(dim, L, seed=77)
    b = orc.Oracle(dim, L, seed=77)
    a.sweep(beta, 3, tile, k)
    a.sweep(beta, 4, tile, k)
    b.sweep(beta, 7, tile, k)
    assert state(a) == state(b)
    assert a.counter == b.counter == 7 * k
    c = orc.Oracle(dim, L, seed=78)
    c.sweep(beta, 7, tile, k)
    assert state(c)[2] != state(a)[2]
    # resume from a checkpoint: spins + counter are the whole state (RNG is stateless)
    d = orc.Oracle(dim, L, seed=77)
    d.sweep(beta, 3, tile, k)
    e = orc.Oracle(dim, L, seed=77)
    e.set_spins(d.spins())
    e.counter = d.counter
    e.sweep(beta, 4, tile, k)
    assert state(e) == state(a)


def test_series_equals_observables_after_each_pass(orc):
    a = orc.Oracle(2, 8, seed=5)
    b = orc.Oracle(2, 8, seed=5)
    E, M = a.sweep_series(BETA_C, 6, 4, 2)
    for p in range(6):
        b.sweep(BETA_C, 1, 4, 2)
        assert state(b)[:2] == (int(E[p, 0]), int(M[p, 0]))


@pytest.mark.parametrize("dim,L,tile,k", [(2, 16, 4, 2), (2, 24, 6, 1), (3, 8, 2, 2)])
def test_tile_order_is_irrelevant(orc, dim, L, tile, k):
    """Tiles of one coarse colour are independent: visiting them in reverse order
    gives the same bits.  Fails if the coarse colouring lets two updated tiles touch."""
    a = orc.Oracle(dim, L, seed=9)
    b = orc.Oracle(dim, L, seed=9)
    b.set_tile_order(True)
    a.sweep(0.35, 5, tile, k)
    b.sweep(0.35, 5, tile, k)
    assert state(a) == state(b)


def test_tile_size_changes_the_trajectory_but_k1_full_tile_is_plain(orc):
    """SURVEY §8(c) reading 5: double checkerboard with k=1 is a different (valid) chain than
    the plain checkerboard; tile = L and tile = 0 are the same thing."""
    a = orc.Oracle(2, 16, seed=4); a.sweep(BETA_C, 3, 16, 1)
    b = orc.Oracle(2, 16, seed=4); b.sweep(BETA_C, 3, 0, 1)
    c = orc.Oracle(2, 16, seed=4); c.sweep(BETA_C, 3, 4, 1)
    assert state(a) == state(b)
    assert state(a)[2] != state(c)[2]


def _site_random(orc, rng, dim, L, i, H, seed):
    """r(i, H) of DESIGN.md §3 R6, restated from the text on top of the KAT-pinned Philox."""
    key, Hw = [seed & 0xFFFFFFFF, seed >> 32], [H & 0xFFFFFFFF, H >> 32]
    if rng == "words":                       # S8c.3
        p = i >> 1
        return orc.philox4x32_10([p >> 2, 0] + Hw, key)[p & 3]
    x, y, z = i % L, (i // L) % L, i // (L * L)
    BW, BH = (16, 2) if dim == 2 else (4, 8)
    px = x >> 1
    GW, GH = -(-(L // 2) // BW), -(-L // BH)
    j = (y % BH) * BW + px % BW
    g = (z * GH + y // BH) * GW + px // BW
    head = 0
    for q in range(12):                      # plane 0 is the most significant bit
        plane = orc.philox4x32_10([g, 3 + 256 * (q >> 2)] + Hw, key)[q & 3]
        head = (head << 1) | ((plane >> j) & 1)
    tail = orc.philox4x32_10([i >> 1, 4] + Hw, key)[0] >> 12
    return (head << 20) | tail


@pytest.mark.parametrize("dim,L", [(2, 8), (2, 36), (3, 4), (3, 10)])
def test_plain_checkerboard_against_lattice_synchronous_numpy(orc, both_rngs, dim, L):
    """tile = L, J = +1: one half-sweep is a synchronous update of one colour.  Restated with
    whole-array numpy operations; the random of every site is rebuilt here from the text of
    the mapping (words: S8c.3; planes: block/bit geometry, 12 plane bits + 20 tail bits) using
    only the oracle's Philox block function, which the KATs pin."""
    seed, beta = 13 + (1 << 40), 0.37 if dim == 2 else 0.2
    o = orc.Oracle(dim, L, seed=seed)
    N = L ** dim
    shape = (L,) * dim
    s = o.spins().astype(np.int64).reshape(shape)        # index order: (z,) y, x
    thr = list(orc.thresholds(beta, dim))
    coords = np.indices(shape)
    parity = coords.sum(axis=0) & 1
    for t in range(2):
        for c in (0, 1):
            H = 2 * t + c
            r = np.array([_site_random(orc, both_rngs, dim, L, i, H, seed) for i in range(N)],
                         dtype=np.uint64).reshape(shape)
            nb = sum(np.roll(s, sh, ax) for ax in range(dim) for sh in (1, -1))
            a = s * nb
            t_sel = np.zeros(shape, dtype=np.uint64)
            for m in range(1, dim + 1):
                t_sel = np.where(a == 2 * m, np.uint64(thr[m - 1]), t_sel)
            flip = ((a <= 0) | (r < t_sel)) & (parity == c)
            s = np.where(flip, -s, s)
    o.sweep(beta, 2, L, 1)
    assert np.array_equal(o.spins().astype(np.int64).reshape(shape), s)
    # the exported per-site random agrees with the restatement, memo on or off
    o.set_memo(False)
    for i in (0, 1, N // 2 + 3, N - 1):
        assert o.sweep_random(i, 5) == _site_random(orc, both_rngs, dim, L, i, 5, seed)


def test_plane_randoms_are_distinct_bits(orc):
    """Planes mapping: the 32 sites of a block take different bit positions of the same planes
    and every active site of a half-sweep owns a distinct (block, bit) — no random bit is used
    twice in a half-sweep.  Checked by brute force on small lattices, both dimensions."""
    for dim, L in ((2, 6), (2, 34), (3, 4), (3, 10)):
        N = L ** dim
        BW, BH = (16, 2) if dim == 2 else (4, 8)
        GW, GH = -(-(L // 2) // BW), -(-L // BH)
        for c in (0, 1):
            seen = set()
            for i in range(N):
                x, y, z = i % L, (i // L) % L, i // (L * L)
                if (x + y + z) & 1 != c:
                    continue
                key = ((z * GH + y // BH) * GW + (x >> 1) // BW, (y % BH) * BW + (x >> 1) % BW)
                assert key not in seen and 0 <= key[1] < 32
                seen.add(key)


def test_memo_is_only_a_cache(orc):
    a = orc.Oracle(2, 16, seed=5); b = orc.Oracle(2, 16, seed=5)
    b.set_memo(False)
    a.sweep(BETA_C, 3, 4, 2); b.sweep(BETA_C, 3, 4, 2)
    assert a.hash() == b.hash()


@pytest.mark.parametrize("dim,L,tile,k", [(2, 16, 4, 2), (3, 6, 6, 1)])
def test_z2_symmetry(orc, dim, L, tile, k):
    """Start from -s0 ⇒ trajectory -s_t: same E, opposite M (the update depends on s_i·field)."""
    a = orc.Oracle(dim, L, seed=21)
    b = orc.Oracle(dim, L, seed=21)
    b.set_spins(-a.spins())
    a.sweep(0.3, 6, tile, k)
    b.sweep(0.3, 6, tile, k)
    assert np.array_equal(a.spins(), -b.spins())
    assert state(a)[0] == state(b)[0] and state(a)[1] == -state(b)[1]


@pytest.mark.parametrize("dim,L,tile,k", [(2, 16, 4, 2), (2, 8, 8, 1), (3, 8, 4, 1)])
def test_gauge_invariance_mattis(orc, dim, L, tile, k):
    """J'_d(i) = ε_i ε_(i+e_d) J_d(i), start ε·s0 ⇒ trajectory ε·s_t and the same E series.
    With J = +1 this is the Mattis model: exercises the whole coupling path (forward bond
    J_d(i), back bond J_d(i-e_d), the d-major layout) against the ferromagnet."""
    N = L ** dim
    rng = np.random.default_rng(5)
    eps = (1 - 2 * rng.integers(0, 2, N)).astype(np.int8)
    e = eps.reshape((L,) * dim)
    for J0 in (None, W.couplings(dim, L, 17)):
        Jp = np.empty((dim,) + (L,) * dim, dtype=np.int8)
        for d in range(dim):
            base = 1 if J0 is None else J0.reshape((dim,) + (L,) * dim)[d]
            Jp[d] = e * np.roll(e, -1, axis=dim - 1 - d) * base
        a = orc.Oracle(dim, L, seed=33, J=J0)
        b = orc.Oracle(dim, L, seed=33, J=Jp.reshape(-1))
        b.set_spins(a.spins() * eps)
        Ea, _ = a.sweep_series(0.5, 5, tile, k)
        Eb, _ = b.sweep_series(0.5, 5, tile, k)
        assert np.array_equal(Ea, Eb)
        assert np.array_equal(a.spins() * eps, b.spins())


def test_unit_couplings_equal_null(orc):
    a = orc.Oracle(2, 16, seed=3)
    b = orc.Oracle(2, 16, seed=3, J=np.ones(2 * 256, dtype=np.int8))
    a.sweep(BETA_C, 4, 4, 2)
    b.sweep(BETA_C, 4, 4, 2)
    assert state(a) == state(b)


def test_replicas_are_independent_runs_sharing_J(orc):
    """A batched handle equals R single handles (realisations worked on concurrently)."""
    J = W.couplings(2, 16, 5)
    seeds = [100, 101, 102]
    b = orc.Oracle(2, 16, seeds=seeds, J=J)
    b.sweep(1.0, 5, 4, 4)
    singles = []
    for r, sd in enumerate(seeds):
        o = orc.Oracle(2, 16, seed=sd, J=J)
        o.sweep(1.0, 5, 4, 4)
        assert state(o) == state(b, r)
        singles.append(o.spins().astype(np.int64))
    assert b.overlap(0, 2) == int((singles[0] * singles[2]).sum())
    assert b.overlap(1, 1) == 256


def test_argument_checks(orc):
    o = orc.Oracle(2, 16, seed=1)
    for tile in (3, 5, 16 // 1 + 2, 6):       # odd, not a divisor
        with pytest.raises(ValueError):
            o.sweep(0.4, 1, tile, 1)
    o12 = orc.Oracle(2, 12, seed=1)
    with pytest.raises(ValueError):
        o12.sweep(0.4, 1, 4, 1)               # L/T = 3 odd: periodic coarse colouring impossible
    with pytest.raises(ValueError):
        o.sweep(0.4, 1, 4, 0)
    with pytest.raises(ValueError):
        o.sweep(-1.0, 1, 4, 1)
    with pytest.raises(ValueError):
        orc.Oracle(2, 7, seed=1)
    with pytest.raises(ValueError):
        orc.Oracle(4, 8, seed=1)


def test_hot_start_is_unbiased_and_seeded(orc):
    o = orc.Oracle(2, 256, seed=123456789012345)
    s = o.spins().astype(np.int64)
    assert abs(s.sum()) < 5 * 256
    assert abs((s[:-1] * s[1:]).sum()) < 5 * 256
    assert not np.array_equal(s, orc.Oracle(2, 256, seed=123456789012346).spins())
    # hi word of the seed is part of the key
    assert not np.array_equal(orc.Oracle(2, 8, seed=1).spins(), orc.Oracle(2, 8, seed=1 + 2 ** 32).spins())


def test_multi_realisation_batch_is_R_ordinary_runs_with_a_shared_random_stream(orc, both_rngs):
    """Asynchronous multi-spin coding batch (R17): realisation r of a multi batch = an ordinary
    single run with couplings J[r], started from the hot start of seeds[r], whose sweep key is the shared one."""
    dim, L, R, K = 2, 16, 3, 777
    Js = np.stack([W.couplings(dim, L, 50 + r) for r in range(R)])
    seeds = [11, 12, 13]
    m = orc.Oracle(dim, L, seeds=seeds, J=Js, sweep_seed=K)
    m.sweep(0.9, 4, 4, 2)
    for r in range(R):
        start = orc.Oracle(dim, L, seed=seeds[r]).spins()                 # hot start of seeds[r]
        single = orc.Oracle(dim, L, seed=K, J=Js[r])                      # sweep key K, couplings J[r]
        single.set_spins(start)
        single.sweep(0.9, 4, 4, 2)
        assert np.array_equal(m.spins()[r], single.spins())
        assert int(m.observables()[0][r]) == int(single.observables()[0][0])
    # shared randoms: the same site of two realisations sees the same r(i, H)
    assert m.sweep_random(5, 3, r=0) == m.sweep_random(5, 3, r=2)
