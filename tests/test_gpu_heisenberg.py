"""GPU parity of the Heisenberg path (include/heisenberg.h) against oracle/heisenberg_oracle.cpp: single
precision with every operation fixed (readings H1-H8), so the bar is bit-exact spins; E and M are sums whose order
is free and are compared to double rounding."""
import numpy as np
import pytest

from oracle import heisenberg as HO

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1006_3865_b200 as pkg
    pkg.use_torch()
    return pkg


def _same(g, o):
    sg = np.asarray(g.copy_spins()).view(np.uint32).reshape(3, -1)
    so = o.spins().view(np.uint32)
    bad = np.flatnonzero((sg != so).any(axis=0))
    assert bad.size == 0, f"{bad.size} spins differ bitwise, first sites {bad[:8]}"
    Eg, Mg = g.observables()
    Eo, Mo = o.observables()
    tol = 1e-9 * g.dim * g.N
    assert abs(Eg - Eo) <= tol and np.all(np.abs(Mg - Mo) <= tol)


@pytest.mark.parametrize("dim,L,seed", [(2, 2, 1), (2, 64, 2), (2, 250, 3), (3, 2, 4), (3, 8, 5), (3, 30, 6)])
def test_hot_start(P, dim, L, seed):
    _same(P.Heisenberg(dim, L, seed=seed), HO.HeisenbergOracle(dim, L, seed=seed))


# dim, L, tile, k, n, beta, expected path
CASES = [
    (2, 2, 2, 1, 4, 0.7, "heis_generic"),
    (2, 12, 6, 2, 3, 0.7, "heis_generic"),          # tile without a staged kernel
    (2, 20, 10, 1, 3, 1.5, "heis_generic"),
    (2, 64, 64, 2, 3, 0.7, "heis_generic"),         # T = L: plain checkerboard
    (2, 64, 0, 1, 3, 0.7, "heis_generic"),
    (2, 64, 16, 1, 3, 0.7, "heis_tile"),
    (2, 64, 16, 3, 2, 2.0, "heis_tile"),
    (2, 64, 32, 2, 3, 0.7, "heis_tile"),
    (2, 128, 64, 2, 2, 1.2, "heis_tile"),
    (2, 192, 32, 1, 3, 0.0, "heis_tile"),           # beta = 0: everything accepted; 6 x 6 tiles
    (2, 192, 16, 2, 2, 50.0, "heis_tile"),          # cold: P underflows to 0 for most moves
    (2, 320, 32, 4, 2, 0.9, "heis_tile"),           # several tiles, ragged against the 148-SM grid
    (2, 256, 64, 1, 3, 0.7, "heis_tile"),
    (3, 2, 2, 1, 3, 0.6, "heis_generic"),
    (3, 12, 6, 2, 2, 0.6, "heis_generic"),
    (3, 16, 16, 1, 2, 0.693, "heis_generic"),
    (3, 8, 4, 2, 3, 0.693, "heis_tile"),
    (3, 16, 8, 2, 2, 0.693, "heis_tile"),
    (3, 32, 8, 1, 2, 0.693, "heis_tile"),
    (3, 32, 16, 2, 2, 0.4, "heis_tile"),
    (3, 48, 8, 3, 1, 5.0, "heis_tile"),
    (3, 24, 4, 1, 2, 0.693, "heis_tile"),
]


@pytest.mark.parametrize("dim,L,T,k,n,beta,path", CASES)
def test_sweep_parity(P, dim, L, T, k, n, beta, path):
    g = P.Heisenberg(dim, L, seed=7)
    o = HO.HeisenbergOracle(dim, L, seed=7)
    g.sweep(beta, n, T, k)
    o.sweep(beta, n, T, k)
    assert g.sweep_path() == path
    assert g.counter == o.counter == n * k
    _same(g, o)


@pytest.mark.parametrize("dim,L,T,k", [(2, 64, 32, 2), (2, 128, 64, 1), (3, 16, 8, 2)])
def test_tile_and_generic_kernels_agree(P, dim, L, T, k):
    a, b = P.Heisenberg(dim, L, seed=9), P.Heisenberg(dim, L, seed=9)
    b.force_generic(True)
    a.sweep(0.8, 3, T, k); b.sweep(0.8, 3, T, k)
    assert a.sweep_path() == "heis_tile" and b.sweep_path() == "heis_generic"
    assert np.array_equal(np.asarray(a.copy_spins()).view(np.uint32), np.asarray(b.copy_spins()).view(np.uint32))


def test_sweeps_compose_and_counter_resume(P):
    a, b = P.Heisenberg(2, 128, seed=4), P.Heisenberg(2, 128, seed=4)
    a.sweep(0.9, 5, 32, 2)
    b.sweep(0.9, 2, 32, 2); b.sweep(0.9, 3, 32, 2)
    assert np.array_equal(np.asarray(a.copy_spins()), np.asarray(b.copy_spins()))
    # resume from a copy: set_spins + set_counter reproduce the continuation
    c = P.Heisenberg(2, 128, seed=4)
    c.set_spins(np.asarray(a.copy_spins())); c.counter = a.counter
    a.sweep(0.9, 2, 32, 2); c.sweep(0.9, 2, 32, 2)
    assert np.array_equal(np.asarray(a.copy_spins()), np.asarray(c.copy_spins()))


@pytest.mark.parametrize("dim,L,T,k,n", [(2, 64, 32, 2, 5), (3, 16, 8, 1, 4), (2, 24, 12, 1, 3)])
def test_sweep_series(P, dim, L, T, k, n):
    """heis_sweep_series: E and M after every pass equal the oracle's observables after the same passes."""
    import torch
    g, o = P.Heisenberg(dim, L, seed=13), HO.HeisenbergOracle(dim, L, seed=13)
    Eg, Mg = g.sweep_series(0.8, n, T, k)
    tol = 1e-9 * dim * L ** dim
    for p in range(n):
        o.sweep(0.8, 1, T, k)
        Eo, Mo = o.observables()
        assert abs(Eg[p] - Eo) <= tol and np.all(np.abs(Mg[p] - Mo) <= tol)
    _same(g, o)
    Ed = torch.zeros(n, dtype=torch.float64, device="cuda")          # device buffer, E only
    g.sweep_series(0.8, n, T, k, E=Ed, M=None)
    o.sweep(0.8, n, T, k)
    assert abs(float(Ed[-1].item()) - o.observables()[0]) <= tol
    _same(g, o)


def test_set_spins_then_sweep_matches_oracle(P):
    rs = np.random.RandomState(3)
    v = rs.normal(size=(3, 64 * 64)).astype(np.float32)
    v /= np.linalg.norm(v, axis=0, keepdims=True).astype(np.float32)
    g, o = P.Heisenberg(2, 64, seed=1), HO.HeisenbergOracle(2, 64, seed=1)
    g.set_spins(v); o.set_spins(v)
    g.sweep(1.0, 3, 32, 2); o.sweep(1.0, 3, 32, 2)
    _same(g, o)


def test_device_buffers(P):
    import torch
    g, o = P.Heisenberg(2, 64, seed=12), HO.HeisenbergOracle(2, 64, seed=12)
    g.sweep(0.7, 2, 32, 1); o.sweep(0.7, 2, 32, 1)
    d = torch.empty(3 * 64 * 64, dtype=torch.float32, device="cuda")
    g.copy_spins(d)
    assert np.array_equal(d.cpu().numpy().view(np.uint32).reshape(3, -1), o.spins().view(np.uint32))


def test_full_size_sampled_against_the_oracle(P):
    """bench.py --heisenberg launch configuration (2D L=4096, tile 32, k=4; 3D L=256 tile 8): the oracle recomputes
    single tiles from the GPU's own previous state — every update of a tile depends only on the tile and its halo."""
    for dim, L, T, k in ((2, 4096, 32, 4), (3, 256, 8, 2)):
        g = P.Heisenberg(dim, L, seed=3)
        g.sweep(0.693, 2, T, k)
        before = np.asarray(g.copy_spins()).reshape((3,) + (L,) * dim).copy()
        t0 = g.counter
        g.sweep(0.693, 1, T, k)
        after = np.asarray(g.copy_spins()).reshape((3,) + (L,) * dim)
        s = np.linalg.norm(after.reshape(3, -1)[:, ::977].astype(np.float64), axis=0)
        assert np.max(np.abs(s - 1.0)) < 6e-7
        # a window of 4 tiles per axis around a few tile positions, run as its own small periodic lattice is NOT
        # the same problem (different site indices -> different random numbers), so compare through the generic kernel
        h = P.Heisenberg(dim, L, seed=3)
        h.force_generic(True)
        h.set_spins(before.reshape(3, -1)); h.counter = t0
        h.sweep(0.693, 1, T, k)
        assert h.sweep_path() == "heis_generic"
        assert np.array_equal(np.asarray(h.copy_spins()).view(np.uint32), after.reshape(3, -1).view(np.uint32))
        g.destroy(); h.destroy()


def test_full_size_first_pass_rows_against_the_oracle(P):
    """2D L=4096 (the bench size): the oracle runs the full lattice for one pass (16.7 M updates, seconds)."""
    L, T, k = 4096, 32, 1
    g, o = P.Heisenberg(2, L, seed=3), HO.HeisenbergOracle(2, L, seed=3)
    g.sweep(0.693, 1, T, k); o.sweep(0.693, 1, T, k)
    _same(g, o)


def test_errors(P):
    g = P.Heisenberg(2, 64, seed=1)
    for bad in ((0.5, 1, 5, 1), (0.5, 1, 64 // 3, 1), (0.5, 1, 32, 0), (-0.1, 1, 32, 1), (float("nan"), 1, 32, 1), (0.5, -1, 32, 1)):
        with pytest.raises(P.IsingError):
            g.sweep(*bad)
    with pytest.raises(P.IsingError):
        P.Heisenberg(2, 63)
    with pytest.raises(P.IsingError):
        P.Heisenberg(4, 8)
