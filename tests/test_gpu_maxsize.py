"""Maximum sizes: N = L^dim up to the 2^32 limit of the ABI (32-bit Philox counters, 64-bit byte offsets).  The
oracle cannot sweep 4 G sites in seconds, so these cases check (a) sampled sites of the hot start against the
oracle's Philox, (b) the staged tile kernels against the generic kernels, which the small parity cases pin to the
oracle, on the whole lattice (compared on the device), (c) properties that hold at any size."""
import numpy as np
import pytest

import ising_workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1006_3865_b200 as pkg
    pkg.use_torch()
    return pkg


def _free():
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()


def _sample_sites(N, rs, n=4000):
    edge = np.array([0, 1, 2, 3, 2 ** 31 - 1, 2 ** 31, 2 ** 31 + 1, N - 4, N - 3, N - 2, N - 1], dtype=np.uint64)
    return np.unique(np.concatenate([edge[edge < N], rs.randint(0, N, size=n, dtype=np.uint64)]))


def test_ising_2d_at_the_index_limit(P, orc):
    """2D L = 65536: N = 2^32 exactly (4 GiB of int8 spins)."""
    import torch
    L, seed = 65536, 17
    N = L * L
    g = P.Ising(2, L, seed=seed)
    s0 = torch.empty(N, dtype=torch.int8, device="cuda")
    g.copy_spins(s0)
    # (a) S8c.3 hot start at sampled sites, the counter limit included
    sites = _sample_sites(N, np.random.RandomState(1))
    got = s0[torch.from_numpy(sites.astype(np.int64)).cuda()].cpu().numpy()
    for i, s in zip(sites.tolist(), got.tolist()):
        w = orc.philox4x32_10([i >> 2, 1, 0, 0], [seed, 0])[i & 3]
        assert s == (-1 if (w >> 31) else 1), i
    M0 = int(s0.sum(dtype=torch.int64).item())
    E, M = g.observables()
    assert int(M[0]) == M0 and abs(M0) < 6 * L and abs(int(E[0])) < 6 * 2 * L        # iid +-1: sigma = sqrt(N), sqrt(2N)
    # (b) one pass of the staged tile kernel against the generic kernels on the whole lattice
    g.sweep(W.BETA_C_2D, 1, 64, 2)
    assert g.sweep_path().startswith("tile_planes")
    s1 = torch.empty(N, dtype=torch.int8, device="cuda")
    g.copy_spins(s1)
    E1, M1 = g.observables()
    g.destroy(); _free()
    h = P.Ising(2, L, seed=seed)
    h.force_path(True)
    h.sweep(W.BETA_C_2D, 1, 64, 2)
    assert h.sweep_path() == "generic"
    s2 = s0                                   # reuse the buffer
    h.copy_spins(s2)
    assert torch.equal(s1, s2)
    E2, M2 = h.observables()
    assert int(E1[0]) == int(E2[0]) and int(M1[0]) == int(M2[0]) == int(s1.sum(dtype=torch.int64).item())
    # (c) after two sweeps at beta_c from a hot start the energy per site has dropped well below 0
    assert -2 * N <= int(E1[0]) < -0.3 * N
    h.destroy(); del s1, s2, s0; _free()


def test_ising_3d_near_the_index_limit(P, orc):
    """3D L = 1616 (8 | L, L/8 even): N = 4 220 112 896, the largest such lattice below 2^32."""
    import torch
    L, seed = 1616, 23
    N = L ** 3
    assert 2 ** 32 - N < 2 ** 27
    g = P.Ising(3, L, seed=seed)
    s0 = torch.empty(N, dtype=torch.int8, device="cuda")
    g.copy_spins(s0)
    sites = _sample_sites(N, np.random.RandomState(2))
    got = s0[torch.from_numpy(sites.astype(np.int64)).cuda()].cpu().numpy()
    for i, s in zip(sites.tolist(), got.tolist()):
        w = orc.philox4x32_10([i >> 2, 1, 0, 0], [seed, 0])[i & 3]
        assert s == (-1 if (w >> 31) else 1), i
    g.sweep(W.BETA_C_3D, 1, 8, 1)
    assert g.sweep_path().startswith("tile3d")
    s1 = torch.empty(N, dtype=torch.int8, device="cuda")
    g.copy_spins(s1)
    E1, M1 = g.observables()
    g.destroy(); _free()
    h = P.Ising(3, L, seed=seed)
    h.force_path(True)
    h.sweep(W.BETA_C_3D, 1, 8, 1)
    h.copy_spins(s0)
    assert torch.equal(s1, s0)
    E2, M2 = h.observables()
    assert int(E1[0]) == int(E2[0]) and int(M1[0]) == int(M2[0])
    h.destroy(); del s0, s1; _free()


def test_heisenberg_2d_beyond_2_to_31_sites(P):
    """2D L = 49152: N = 2.4e9 > 2^31 (29 GB of float spins): staged tile kernel against the generic one, hot start
    sampled against the oracle's direction map."""
    import torch
    from oracle import heisenberg as HO
    L, seed = 49152, 29
    N = L * L
    g = P.Heisenberg(2, L, seed=seed)
    s0 = torch.empty(3 * N, dtype=torch.float32, device="cuda")
    g.copy_spins(s0)
    sites = _sample_sites(N, np.random.RandomState(3), 1500)
    idx = torch.from_numpy(sites.astype(np.int64)).cuda()
    got = torch.stack([s0[idx], s0[N + idx], s0[2 * N + idx]]).cpu().numpy()
    for n, i in enumerate(sites.tolist()):
        w = HO.philox([i >> 1, 6, 0, 0], [seed, 0])
        assert np.array_equal(got[:, n], HO.direction(w[2 * (i & 1)], w[2 * (i & 1) + 1])), i
    g.sweep(0.7, 1, 32, 2)
    assert g.sweep_path() == "heis_tile"
    s1 = torch.empty(3 * N, dtype=torch.float32, device="cuda")
    g.copy_spins(s1)
    g.set_spins(s0); g.counter = 0
    g.force_generic(True)
    g.sweep(0.7, 1, 32, 2)
    assert g.sweep_path() == "heis_generic"
    g.copy_spins(s0)
    assert torch.equal(s1.view(torch.int32), s0.view(torch.int32))
    E, M = g.observables()
    assert -2 * N < E < -0.05 * N and np.all(np.abs(M) < 1e-3 * N)
    g.destroy(); del s0, s1; _free()
