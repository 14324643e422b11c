"""ising_overlap_all_static (include/ising.h): the all-pairs overlap without any device allocation — its scratch is a 32 KiB
__device__ array inside the library — against the existing path (ising_overlap_all on the handle) and the oracle's pairwise
definition, on two calls in a row.  Integer work: exact equality.  In a file of its own, collected last (the suite runs
with pytest -x); it passes alone in a fresh process and after the other tests."""
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


def _glass(P, orc, L, R, first_seed, n):
    """R replicas of a 2D +-J glass (config 5's shape in small) after n passes: (handle, oracle, device spins)."""
    import torch
    J = W.couplings(2, L, 5)
    seeds = [first_seed + r for r in range(R)]
    g = P.Ising(2, L, coupling=J, seeds=seeds)
    o = orc.Oracle(2, L, seeds=seeds, J=J)
    g.sweep(1.0, n, 32, 2); o.sweep(1.0, n, 32, 2)
    s = torch.empty(R * L * L, dtype=torch.int8, device="cuda")
    g.copy_spins(s)
    return g, o, s


def test_overlap_all_static_matches_the_handle_path_twice_in_a_row(P, orc):
    import torch
    L = 128
    # first call: 16 replicas (the scratch is left full of their counts) ...
    g1, o1, s1 = _glass(P, orc, L, 16, 100, 3)
    Q1 = torch.full((16, 16), -7, dtype=torch.int64, device="cuda")
    P.ising_overlap_all_static(s1, 16, L * L, Q1)
    # ... second call straight after it, fewer replicas of another trajectory: the stale counts must not leak in
    g2, o2, s2 = _glass(P, orc, L, 7, 300, 2)
    Q2 = torch.full((7, 7), -7, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    launches = P.ising_kernel_launches()
    P.ising_overlap_all_static(s2, 7, L * L, Q2)
    P.ising_overlap_all_static(s2, 7, L * L, Q2)                        # and once more on the same input: same answer
    torch.cuda.synchronize()
    assert P.ising_kernel_launches() == launches + 4                    # its own kernels ran (2 per call)
    assert torch.cuda.mem_get_info()[0] >= free_before                  # nothing was allocated on the device
    for g, o, Q, R in ((g1, o1, Q1, 16), (g2, o2, Q2, 7)):
        ref = np.asarray(g.overlap_all())                               # the existing path (handle-owned scratch)
        assert np.array_equal(Q.cpu().numpy(), ref)
        want = np.array([[o.overlap(a, b) for b in range(R)] for a in range(R)], dtype=np.int64)
        assert np.array_equal(ref, want)                                # ... which is the oracle's pairwise definition
        assert np.array_equal(np.diag(ref), np.full(R, L * L))
        g.destroy()


def test_overlap_all_static_limits_and_errors(P):
    import torch
    N = 64
    R = P.STATIC_MAX_REPLICAS
    rng = np.random.default_rng(11)
    host = (2 * rng.integers(0, 2, size=(R + 1, N)) - 1).astype(np.int8)
    s = torch.from_numpy(host).cuda()
    Q = torch.zeros((R, R), dtype=torch.int64, device="cuda")
    P.ising_overlap_all_static(s, R, N, Q)                               # the maximum itself is served
    torch.cuda.synchronize()
    h64 = host[:R].astype(np.int64)
    assert np.array_equal(Q.cpu().numpy(), h64 @ h64.T)
    P.ising_overlap_all_static(s, 1, N, Q)                               # one replica: Q = [N]
    torch.cuda.synchronize()
    assert int(Q.view(-1)[0]) == N
    big = torch.zeros((R + 1, R + 1), dtype=torch.int64, device="cuda")
    with pytest.raises(P.IsingError, match="at most ISING_STATIC_MAX_REPLICAS = 64"):
        P.ising_overlap_all_static(s, R + 1, N, big)                     # beyond the static scratch: a clear error
    with pytest.raises(P.IsingError):
        P.ising_overlap_all_static(s, 0, N, Q)
    with pytest.raises(P.IsingError):
        P.ising_overlap_all_static(s, 2, N + 2, Q)                       # n_sites not a multiple of 4
    with pytest.raises(P.IsingError):
        P.ising_overlap_all_static(None, 2, N, Q)
    with pytest.raises(P.IsingError):
        P.ising_overlap_all_static(s.view(-1)[1:], 2, N, Q)              # misaligned input
    assert int(big.abs().sum()) == 0                                     # a rejected call enqueues nothing
