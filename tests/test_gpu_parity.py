"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit, on the
same seeded inputs.  Integer work only, so the bar is exact equality of every spin, E and M."""
import numpy as np
import pytest

import ising_workloads as W

pytestmark = pytest.mark.gpu

BC2, BC3 = W.BETA_C_2D, W.BETA_C_3D


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1006_3865_b200 as pkg
    pkg.use_torch()
    return pkg


RNGS = ["planes", "words"]


def _both(P, orc, dim, L, seeds, J=None, rng="planes"):
    g = P.Ising(dim, L, coupling=J, seeds=seeds, rng=rng)
    o = orc.Oracle(dim, L, seeds=seeds, J=J, rng=rng)
    return g, o


def _same_state(g, o):
    sg = np.asarray(g.copy_spins()).reshape(-1)
    so = np.asarray(o.spins()).reshape(-1)
    bad = np.flatnonzero(sg != so)
    assert bad.size == 0, f"{bad.size} spins differ, first at {bad[:8]}"
    Eg, Mg = g.observables()
    Eo, Mo = o.observables()
    assert list(Eg) == list(Eo) and list(Mg) == list(Mo)


@pytest.mark.parametrize("dim,L,seed", [(2, 2, 5), (2, 4, 3), (2, 64, 1), (2, 250, 8), (3, 2, 1), (3, 8, 4), (3, 30, 2)])
def test_hot_start(P, orc, dim, L, seed):
    g, o = _both(P, orc, dim, L, [seed])
    _same_state(g, o)


GENERIC = [
    # dim, L, tile, k, n, beta, seeds, jseed
    (2, 2, 2, 1, 5, BC2, [1], None),
    (2, 4, 2, 3, 5, BC2, [3], None),
    (2, 8, 4, 2, 3, BC2, [7], None),
    (2, 64, 0, 1, 20, BC2, [1], None),          # config 1 shape: plain checkerboard
    (2, 64, 8, 4, 6, BC2, [9], None),
    (2, 96, 16, 2, 4, 0.6, [11], None),
    (2, 36, 6, 2, 4, 0.3, [12], None),          # tile not a multiple of 8
    (3, 2, 2, 1, 4, BC3, [2], None),
    (3, 8, 4, 2, 5, BC3, [4], None),            # config 4 shape, small
    (3, 16, 8, 4, 2, BC3, [4], None),
    (3, 12, 6, 1, 3, 0.5, [6], None),
    (2, 16, 4, 4, 10, 1.0, [100], 5),           # config 5 shape, small
    (2, 64, 32, 4, 4, 1.0, [100, 101, 114], 5), # replicas sharing J
    (3, 8, 4, 2, 3, 0.9, [1, 2], 17),
    (2, 32, 8, 1, 3, 0.0, [4], None),           # beta = 0: thresholds are 2^32
    (2, 32, 8, 2, 3, 30.0, [4], None),          # thresholds underflow to 0
]


@pytest.mark.parametrize("rng", RNGS)
@pytest.mark.parametrize("dim,L,tile,k,n,beta,seeds,jseed", GENERIC)
def test_generic_path_matches_oracle(P, orc, dim, L, tile, k, n, beta, seeds, jseed, rng):
    J = W.couplings(dim, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, dim, L, seeds, J, rng)
    g.force_path(True)
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert g.sweep_path() == "generic"
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    assert g.counter == o.counter == n * k
    if len(seeds) > 1:
        assert g.overlap(0, 1) == o.overlap(0, 1)


TILED = [
    # L, tile, k, n, beta, seeds  — several tiles, both tile sizes, wrap-around in both directions
    (64, 32, 1, 3, BC2, [3]),
    (128, 32, 4, 3, BC2, [3]),
    (128, 64, 1, 3, BC2, [5]),
    (256, 64, 4, 2, 0.6, [6]),
    (192, 32, 2, 3, 0.3, [7]),       # B = 6: ragged against the 2-tiles-per-warp job
    (384, 64, 1, 2, BC2, [8]),       # B = 6
    (256, 32, 16, 1, BC2, [3]),
    (128, 32, 2, 2, 0.0, [2]),
    (128, 64, 2, 2, 30.0, [2]),
    (128, 32, 2, 3, BC2, [21, 22, 23]),   # replicas
]


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds", TILED + [(512, 64, 3, 4, 1.0, [31]), (512, 32, 1, 6, 0.2, [32])])
def test_tile_planes_path_matches_oracle(P, orc, L, tile, k, n, beta, seeds, layout):
    """Multi-spin tile kernel (RNG mapping planes), both HBM layouts.  L >= 256 at beta_c draws
    the per-site tail (head == threshold head, probability 2^-12 per site) several times."""
    g, o = _both(P, orc, 2, L, seeds, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.force_path(2)            # a launch per coarse colour also where the cluster-resident kernel would serve
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    assert g.sweep_path() == f"tile_planes_{'i8' if layout == 'int8' else 'bits'}"
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds,jseed", [
    (128, 32, 4, 3, 1.0, [100, 101, 102], 5),      # config 5 shape: +-J glass, replicas share J
    (256, 64, 2, 3, 0.8, [7], 11),
    (192, 32, 1, 4, 0.5, [8, 9], 12),
    (256, 32, 3, 2, 0.0, [3], 13),
])
def test_tile_planes_couplings_match_oracle(P, orc, L, tile, k, n, beta, seeds, jseed, layout):
    """a9 on the multi-spin tile kernel: quenched +-J bonds as bit records shared by the replicas."""
    J = W.couplings(2, L, jseed)
    g, o = _both(P, orc, 2, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.force_path(2)            # a launch per coarse colour (the cluster-resident kernel has its own test)
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    assert g.sweep_path() == f"tile_planes_{'i8' if layout == 'int8' else 'bits'}"
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    if len(seeds) > 1:
        assert g.overlap(0, 1) == o.overlap(0, 1)
    # gauge invariance on the GPU path alone: J' = eps_i eps_j J, s' = eps s gives the same E series
    rng = np.random.default_rng(jseed)
    eps = (1 - 2 * rng.integers(0, 2, size=(L, L))).astype(np.int8)
    Jg = J.reshape(2, L, L) * eps[None] * np.stack([np.roll(eps, -1, 1), np.roll(eps, -1, 0)])
    a = P.Ising(2, L, coupling=J, seeds=seeds[:1]); b = P.Ising(2, L, coupling=Jg.reshape(-1).astype(np.int8), seeds=seeds[:1])
    b.set_spins((a.copy_spins().reshape(L, L) * eps).reshape(-1))
    Ea, _ = a.sweep_series(beta, 2, tile, k); Eb, _ = b.sweep_series(beta, 2, tile, k)
    assert np.array_equal(Ea, Eb)
    assert np.array_equal(a.copy_spins().reshape(L, L) * eps, b.copy_spins().reshape(L, L))


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,k,n,beta,seeds", [
    (16, 1, 4, BC3, [4]),            # B = 2: every halo wraps onto the other tile
    (32, 4, 3, BC3, [4]),            # config 4 shape
    (48, 2, 3, 0.3, [5, 6]),         # B = 6, replicas
    (64, 1, 3, BC3, [9]),            # 2^18 sites: the tail is drawn about 50 times per half-sweep
    (32, 2, 2, 0.0, [2]),
    (32, 2, 2, 9.0, [2]),
])
def test_tile3d_path_matches_oracle(P, orc, L, k, n, beta, seeds, layout):
    """3D 8x8x8 tile kernel (config 4), both HBM layouts, against the oracle."""
    g, o = _both(P, orc, 3, L, seeds, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.force_path(2)            # a launch per colour; E and M by k_observables3d on the records
    Eg, Mg = g.sweep_series(beta, n, 8, k)
    assert g.sweep_path() == f"tile3d_planes_{'i8' if layout == 'int8' else 'bits'}"
    Eo, Mo = o.sweep_series(beta, n, 8, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("k,n,beta,seeds,jseed", [(1, 50, BC2, [1], None), (3, 7, 0.6, [1, 2, 3], None), (2, 9, 1.0, [5, 6], 7),
                                                    (1, 4, 0.0, [2], None)])
def test_plain64_path_matches_oracle(P, orc, k, n, beta, seeds, jseed, layout):
    """a8 / config 1 shape: 64x64 plain checkerboard, all passes in one launch, E and M measured in the kernel."""
    J = W.couplings(2, 64, jseed) if jseed is not None else None
    g, o = _both(P, orc, 2, 64, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    Eg, Mg = g.sweep_series(beta, n, 0, k)
    assert g.sweep_path() == f"plain64_planes_{'i8' if layout == 'int8' else 'bits'}"
    Eo, Mo = o.sweep_series(beta, n, 64, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.sweep(beta, 3, 64, k); o.sweep(beta, 3, 0, k)          # without the series, and composing with the counter
    _same_state(g, o)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds,jseed", [
    (256, 64, 2, 3, BC2, [3], None), (256, 32, 3, 2, 0.3, [4, 5], None), (128, 32, 2, 3, 1.0, [6, 7], 5),
    (512, 64, 1, 4, 0.6, [8], None), (128, 64, 2, 2, 30.0, [2], None), (128, 32, 1, 2, 0.0, [2], None),
])
def test_specialised_kernel_matches_oracle(P, orc, L, tile, k, n, beta, seeds, jseed, layout):
    """Run-time specialisation on the threshold head bits (ising_set_jit ON): same trajectory, bit for bit; and the
    pre-compiled kernel (OFF) continues it identically."""
    J = W.couplings(2, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 2, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.set_jit("on")
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    assert g.last_sweep_specialized() == (beta > 0), "NVRTC specialisation was not used (beta = 0 has no thresholds to fold)"
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.set_jit("off")
    g.sweep(beta, 2, tile, k); o.sweep(beta, 2, tile, k)
    assert not g.last_sweep_specialized()
    _same_state(g, o)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,k,n,beta,seeds", [(32, 2, 3, BC3, [4]), (48, 1, 3, 0.3, [5, 6]), (64, 1, 2, BC3, [9]), (32, 2, 2, 9.0, [2])])
def test_specialised_3d_kernel_matches_oracle(P, orc, L, k, n, beta, seeds, layout):
    """The 3D kernel specialised at run time on its three threshold heads, against the oracle."""
    g, o = _both(P, orc, 3, L, seeds, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.set_jit("on")
    Eg, Mg = g.sweep_series(beta, n, 8, k)
    assert g.last_sweep_specialized()
    Eo, Mo = o.sweep_series(beta, n, 8, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)


@pytest.mark.parametrize("L,tile,k,n,beta,R", [(64, 32, 1, 3, 1.0, 32), (128, 32, 4, 2, 0.8, 16), (128, 64, 2, 3, 1.2, 5),
                                                 (192, 32, 2, 2, 0.5, 32), (128, 64, 1, 2, 0.0, 3), (64, 32, 2, 2, 30.0, 2)])
def test_multi_realisation_batch_matches_oracle(P, orc, L, tile, k, n, beta, R):
    """SURVEY 8(f)-1, asynchronous multi-spin coding (R17): R disorder realisations in one word lattice driven by
    one random stream; every realisation against the oracle's multi batch; and the generic path on the same handle."""
    Js = np.stack([W.couplings(2, L, 900 + r) for r in range(R)])
    seeds = [2000 + r for r in range(R)]
    g = P.Ising(2, L, coupling=Js, seeds=seeds, sweep_seed=4242)
    o = orc.Oracle(2, L, J=Js, seeds=seeds, sweep_seed=4242, rng="words")
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    assert g.sweep_path() == "amsc"
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    assert g.overlap(0, R - 1) == o.overlap(0, R - 1)
    g.force_path(True)                                        # the generic kernels continue the same trajectories
    g.sweep(beta, 1, tile, k); o.sweep(beta, 1, tile, k)
    assert g.sweep_path() == "generic"
    _same_state(g, o)
    g.force_path(False); g.set_rng("planes"); o2 = None       # planes mapping on a multi handle: generic path, still exact
    op = orc.Oracle(2, L, J=Js, seeds=seeds, sweep_seed=4242, rng="planes")
    op.set_spins(o.spins()); op.counter = o.counter
    g.sweep(beta, 1, tile, k); op.sweep(beta, 1, tile, k)
    assert g.sweep_path() == "generic"
    _same_state(g, op)


def test_missing_nvrtc_falls_back_to_the_precompiled_kernel():
    """With libnvrtc unavailable (simulated by ISING_NO_NVRTC in a fresh process) ising_set_jit(ON) still sweeps, on the
    pre-compiled kernel, and still matches the oracle: the fallback is another CUDA kernel, never a CPU path."""
    import os, subprocess, sys
    code = (
        "import numpy as np, paper_1006_3865_b200 as P\n"
        "from oracle import oracle as O\n"
        "P.use_torch()\n"
        "g = P.Ising(2, 128, seed=5); o = O.Oracle(2, 128, seed=5)\n"
        "g.set_jit('on'); g.sweep(0.44, 3, 32, 2); o.sweep(0.44, 3, 32, 2)\n"
        "assert not g.last_sweep_specialized() and g.sweep_path() == 'tile_planes_i8'\n"
        "assert np.array_equal(g.copy_spins(), o.spins())\n"
        "print('fallback ok')\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, ISING_NO_NVRTC="1"),
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0 and "fallback ok" in out.stdout, out.stderr[-2000:]


@pytest.mark.parametrize("L,tile,k,n,beta,seeds", TILED)
def test_tile_i8_path_matches_oracle(P, orc, L, tile, k, n, beta, seeds):
    g, o = _both(P, orc, 2, L, seeds, rng="words")
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    assert g.sweep_path() == ("tile_i8" if beta > 0 else "generic")   # beta = 0: thr = 2^32, generic kernels
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)


def test_paths_agree_and_sweeps_compose(P, orc):
    """sweep(a); sweep(b) == sweep(a+b) across kernel paths and tile sizes (stateless RNG)."""
    a = P.Ising(2, 256, seed=33)
    b = P.Ising(2, 256, seed=33)
    a.sweep(BC2, 2, 32, 4); a.sweep(BC2, 3, 64, 2); a.sweep(BC2, 1, 0, 1)
    b.force_path(True)
    b.sweep(BC2, 2, 32, 4); b.sweep(BC2, 3, 64, 2); b.sweep(BC2, 1, 0, 1)
    assert np.array_equal(a.copy_spins(), b.copy_spins())
    o = orc.Oracle(2, 256, seed=33)
    o.sweep(BC2, 2, 32, 4); o.sweep(BC2, 3, 64, 2); o.sweep(BC2, 1, 0, 1)
    _same_state(a, o)


def test_set_spins_counter_resume_and_invariants(P, orc):
    L = 128
    g = P.Ising(2, L, seed=5)
    up = np.ones(L * L, dtype=np.int8)
    g.set_spins(up)
    E, M = g.observables()
    assert (int(E[0]), int(M[0])) == (-2 * L * L, L * L)          # E(all up) = -2N
    g3 = P.Ising(3, 16, seed=5)
    g3.set_spins(np.ones(16 ** 3, dtype=np.int8))
    assert int(g3.observables()[0][0]) == -3 * 16 ** 3
    with pytest.raises(P.IsingError):
        g.set_spins(np.zeros(L * L, dtype=np.int8))
    # resume: copy state + counter into a fresh handle
    a = P.Ising(2, L, seed=9); a.sweep(BC2, 3, 32, 2)
    b = P.Ising(2, L, seed=9); b.set_spins(a.copy_spins()); b.counter = a.counter
    a.sweep(BC2, 2, 32, 2); b.sweep(BC2, 2, 32, 2)
    assert np.array_equal(a.copy_spins(), b.copy_spins())
    # Z2: start from -s0 gives -s_t
    c = P.Ising(2, L, seed=9); s0 = c.copy_spins().copy()
    d = P.Ising(2, L, seed=9); d.set_spins(-s0)
    c.sweep(0.5, 3, 64, 2); d.sweep(0.5, 3, 64, 2)
    assert np.array_equal(c.copy_spins(), -d.copy_spins())


def test_device_pointer_outputs(P, orc):
    import torch
    g = P.Ising(2, 128, seed=4)
    E = torch.zeros(5, dtype=torch.int64, device="cuda")
    M = torch.zeros(5, dtype=torch.int64, device="cuda")
    g.sweep_series(BC2, 5, 32, 1, E=E, M=M)
    dst = torch.zeros(128 * 128, dtype=torch.int8, device="cuda")
    g.copy_spins(dst)
    o = orc.Oracle(2, 128, seed=4)
    Eo, Mo = o.sweep_series(BC2, 5, 32, 1)
    assert E.cpu().tolist() == Eo[:, 0].tolist() and M.cpu().tolist() == Mo[:, 0].tolist()
    assert np.array_equal(dst.cpu().numpy(), o.spins())


def test_argument_errors(P):
    g = P.Ising(2, 64, seed=1)
    for tile in (3, 5, 48, 128):
        with pytest.raises(P.IsingError):
            g.sweep(0.4, 1, tile, 1)
    with pytest.raises(P.IsingError):
        g.sweep(0.4, 1, 32, 0)
    with pytest.raises(P.IsingError):
        g.sweep(-0.1, 1, 32, 1)
    with pytest.raises(P.IsingError):
        g.sweep(float("nan"), 1, 32, 1)
    with pytest.raises(P.IsingError):
        P.Ising(2, 16, coupling=np.zeros(2 * 256, dtype=np.int8), seed=1)
    g.sweep(0.4, 0, 32, 1)      # zero passes is a no-op
    assert g.counter == 0


@pytest.mark.parametrize("dim,L,T,seeds,layout", [(2, 64, 32, [1], "int8"), (2, 128, 64, [2, 3], "int8"), (2, 128, 64, [4], "bits"),
                                                   (3, 16, 8, [5], "int8"), (2, 8, 4, [6], "int8"), (2, 192, 32, [7], "int8")])
def test_bit_packed_host_io(P, orc, dim, L, T, seeds, layout):
    """ising_copy_spins_bits / ising_set_spins_bits: bit i & 31 of word i >> 5 set <=> s_i = +1, against numpy's packing of
    the oracle's spins; a state set from bits continues like the oracle's."""
    g, o = _both(P, orc, dim, L, seeds)
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(BC2, 2, T, 2); o.sweep(BC2, 2, T, 2)
    want = np.packbits((np.asarray(o.spins()).reshape(-1) > 0).astype(np.uint8), bitorder="little").view(np.uint32)
    got = g.copy_spins_bits()
    assert np.array_equal(got, want)
    # round trip through a fresh handle, then both continue
    h = P.Ising(dim, L, seeds=seeds)
    if layout == "bits":
        h.set_layout(P.ISING_LAYOUT_BITS)
    h.set_spins_bits(got); h.counter = g.counter
    h.sweep(BC2, 2, T, 1); o.sweep(BC2, 2, T, 1)
    _same_state(h, o)
    import torch
    d = torch.zeros(len(seeds) * L ** dim // 32, dtype=torch.int32, device="cuda")
    h.copy_spins_bits(d)
    want = np.packbits((np.asarray(o.spins()).reshape(-1) > 0).astype(np.uint8), bitorder="little").view(np.uint32)
    assert np.array_equal(d.cpu().numpy().view(np.uint32), want)


def test_bit_packed_io_needs_whole_words(P):
    g = P.Ising(2, 6, seed=1)          # N = 36
    with pytest.raises(P.IsingError):
        g.copy_spins_bits(np.zeros(2, dtype=np.uint32))


def test_set_spins_rejects_bad_values_and_keeps_the_state(P, orc):
    """in both situations: state in the canonical array (fresh handle) and state in tile records (after a sweep)"""
    for swept in (False, True):
        g, o = _both(P, orc, 2, 64, [9])
        if swept:
            g.sweep(BC2, 1, 32, 1); o.sweep(BC2, 1, 32, 1)
        bad = np.asarray(o.spins()).reshape(-1).copy()
        bad[1234] = 0
        with pytest.raises(P.IsingError):
            g.set_spins(bad)
        bad[1234] = 3
        bad[-1] = 1
        with pytest.raises(P.IsingError):
            g.set_spins(bad)
        _same_state(g, o)
        g.sweep(BC2, 1, 32, 1); o.sweep(BC2, 1, 32, 1)
        _same_state(g, o)


RESIDENT = [
    # L, tile, k, n, beta, seeds: 1 .. 64 warp jobs per colour, cluster sizes 1 .. 16
    (64, 32, 1, 3, BC2, [3]),
    (128, 64, 2, 4, BC2, [5]),
    (128, 32, 3, 2, 0.6, [4]),
    (192, 32, 2, 3, 0.3, [7]),
    (384, 64, 1, 5, BC2, [8]),
    (256, 32, 2, 4, BC2, [21, 22, 23]),    # one cluster per replica
    (512, 32, 1, 6, 0.2, [32]),
    (512, 64, 3, 2, 1.0, [31]),
    (128, 32, 2, 2, 0.0, [2]),
    (128, 64, 2, 2, 30.0, [2]),
    (448, 32, 2, 2, BC2, [9]),             # B = 14: 49 jobs per colour, ragged against the 64 warps
    (640, 64, 1, 3, BC2, [10]),            # B = 10: 50 jobs
]


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds", RESIDENT)
def test_cluster_resident_kernel_matches_oracle(P, orc, L, tile, k, n, beta, seeds, layout):
    """Small lattices, n >= 2 passes, no series: one launch of one cluster per replica, tiles in registers, boundaries
    through distributed shared memory.  Same trajectory as everything else."""
    g, o = _both(P, orc, 2, L, seeds, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(beta, n, tile, k); o.sweep(beta, n, tile, k)
    assert g.sweep_path() == f"resident_planes_{'i8' if layout == 'int8' else 'bits'}"
    _same_state(g, o)
    if L == 512 and tile == 32 and layout == "int8":                # larger lattices keep the per-pass kernels
        big = P.Ising(2, 1024, seed=1)
        big.sweep(beta, 2, 32, 1)
        assert big.sweep_path() == "grid_planes_i8"             # ... of the grid-resident kernel (test_grid_resident_*)
    g.sweep(beta, 1, tile, k); o.sweep(beta, 1, tile, k)          # a single pass goes through the per-pass kernel and composes
    assert g.sweep_path().startswith("tile_planes")
    g.sweep(beta, 2, tile, k); o.sweep(beta, 2, tile, k)
    _same_state(g, o)
    g.force_path(2)
    g.sweep(beta, 2, tile, k); o.sweep(beta, 2, tile, k)
    assert g.sweep_path().startswith("tile_planes")
    _same_state(g, o)
    g.force_path(0)
    Eg, Mg = g.sweep_series(beta, n + 1, tile, k)                 # E and M after every pass, measured on the registers
    assert g.sweep_path().startswith("resident_planes")
    Eo, Mo = o.sweep_series(beta, n + 1, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    import torch
    Ed = torch.zeros((2, len(seeds)), dtype=torch.int64, device="cuda")   # device buffers, E only
    g.sweep_series(beta, 2, tile, k, E=Ed, M=None)
    Eo, _ = o.sweep_series(beta, 2, tile, k)
    assert np.array_equal(Ed.cpu().numpy(), Eo)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,k,n,beta,seeds", [
    (16, 1, 4, BC3, [4]),            # one job per colour, a cluster of one CTA; every halo wraps onto the other tile
    (32, 4, 3, BC3, [4]),
    (48, 2, 3, 0.3, [5, 6]),         # 27 jobs per colour, two clusters
    (64, 1, 5, BC3, [9]),            # 64 jobs per colour: all 64 warps of a 16-CTA cluster
    (32, 2, 2, 0.0, [2]),
    (32, 2, 2, 9.0, [2]),
])
def test_cluster_resident_3d_kernel_matches_oracle(P, orc, L, k, n, beta, seeds, layout):
    """3D, L <= 64, n >= 2 passes: one launch of one cluster per replica, slices in registers, faces through DSMEM."""
    g, o = _both(P, orc, 3, L, seeds, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(beta, n, 8, k); o.sweep(beta, n, 8, k)
    assert g.sweep_path() == f"resident3d_planes_{'i8' if layout == 'int8' else 'bits'}"
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, 8, k)          # E and M after every pass, counted on the registers
    assert g.sweep_path().startswith("resident3d_planes")
    Eo, Mo = o.sweep_series(beta, n, 8, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    g.sweep(beta, 1, 8, k); o.sweep(beta, 1, 8, k)
    assert g.sweep_path().startswith("tile3d_planes")
    g.sweep(beta, 2, 8, k); o.sweep(beta, 2, 8, k)
    _same_state(g, o)
    if L == 64 and layout == "int8":
        big = P.Ising(3, 128, seed=1)
        big.sweep(beta, 2, 8, 1)
        assert big.sweep_path() == "grid3d_planes_i8"           # larger lattices: the grid-resident kernel (test_grid_resident_3d_*)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds,jseed", [
    (64, 32, 2, 4, 1.0, [100, 101, 102], 5),       # small +-J glass, three replicas = three clusters sharing J
    (128, 64, 1, 3, 0.8, [7], 11),
    (192, 32, 3, 2, 0.5, [8, 9], 12),
    (512, 32, 1, 3, 1.2, [3], 13),
])
def test_cluster_resident_kernel_with_couplings(P, orc, L, tile, k, n, beta, seeds, jseed, layout):
    """a9 on the cluster-resident kernel: the tiles' coupling words stay in registers with the spins."""
    J = W.couplings(2, L, jseed)
    g, o = _both(P, orc, 2, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(beta, n, tile, k); o.sweep(beta, n, tile, k)
    assert g.sweep_path() == f"resident_planes_{'i8' if layout == 'int8' else 'bits'}"
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    assert g.sweep_path().startswith("resident_planes")
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    for a in range(len(seeds)):
        for b in range(a + 1, len(seeds)):
            assert g.overlap(a, b) == o.overlap(a, b)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,k,n,beta,seeds,jseed", [
    (16, 2, 3, 0.9, [1], 3),                 # B = 2
    (32, 1, 3, 1.1, [4, 5, 6], 7),           # 3D Edwards-Anderson glass, replicas share J
    (48, 3, 2, 0.5, [8], 9),
    (96, 1, 2, 0.9, [2], 10),                # B = 12: too large for the resident kernel
    (32, 2, 2, 0.0, [2], 11),
])
def test_tile3d_couplings_match_oracle(P, orc, L, k, n, beta, seeds, jseed, layout):
    """a9 in 3D: quenched +-J bonds as bit records (six words per slice and colour), per-pass and cluster-resident kernels."""
    J = W.couplings(3, L, jseed)
    g, o = _both(P, orc, 3, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.force_path(2)
    Eg, Mg = g.sweep_series(beta, n, 8, k)          # a launch per colour, E and M on the records
    assert g.sweep_path() == f"tile3d_planes_{'i8' if layout == 'int8' else 'bits'}"
    Eo, Mo = o.sweep_series(beta, n, 8, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.force_path(0)
    g.sweep(beta, n, 8, k); o.sweep(beta, n, 8, k)
    assert g.sweep_path().startswith("resident3d_planes" if L <= 64 else "grid3d_planes")
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, 8, k)          # L <= 64: measured on the registers of the resident kernel
    Eo, Mo = o.sweep_series(beta, n, 8, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    for a in range(len(seeds)):
        for b in range(a + 1, len(seeds)):
            assert g.overlap(a, b) == o.overlap(a, b)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,k,n,beta,seeds,jseed", [
    (128, 1, 4, BC2, [3], None),
    (192, 2, 3, 0.3, [7], None),             # 6 x 6 register tiles of 32
    (256, 1, 3, BC2, [21, 22], None),        # replicas
    (512, 2, 2, BC2, [32], None),
    (640, 1, 2, 0.6, [5], None),             # L/32 = 20 tiles: too many jobs at 32, cut into 64 x 64 tiles instead
    (128, 2, 3, 1.0, [100, 101], 5),         # +-J
    (128, 1, 1, BC2, [4], None),             # a single pass too
])
def test_plain_checkerboard_on_the_resident_kernel(P, orc, L, k, n, beta, seeds, jseed, layout):
    """a8 beyond L = 64: tile == L, the whole lattice's even sites, barrier, odd sites, on the cluster-resident kernel."""
    J = W.couplings(2, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 2, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(beta, n, 0, k); o.sweep(beta, n, 0, k)
    assert g.sweep_path() == f"resident_plain_{'i8' if layout == 'int8' else 'bits'}"
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n + 1, L, k)
    assert g.sweep_path().startswith("resident_plain")
    Eo, Mo = o.sweep_series(beta, n + 1, L, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.sweep(beta, 2, 32, 1); o.sweep(beta, 2, 32, 1)      # and back to tiles
    _same_state(g, o)
    g.force_path(True)
    g.sweep(beta, 1, 0, k); o.sweep(beta, 1, 0, k)
    assert g.sweep_path() == "generic"
    _same_state(g, o)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,k,n,beta,seeds,jseed", [
    (1024, 1, 3, BC2, [3], None),
    (704, 2, 2, 0.3, [7, 8], None),          # 22 x 22 tiles of 32 (11 x 11 of 64 would be odd)
    (768, 1, 2, 1.0, [100], 5),              # +-J
])
def test_plain_checkerboard_large_lattices(P, orc, L, k, n, beta, seeds, jseed, layout):
    """a8 for L > 512: the tile kernel with a launch per half-sweep over all tiles."""
    J = W.couplings(2, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 2, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    Eg, Mg = g.sweep_series(beta, n, 0, k)
    assert g.sweep_path() == f"tile_plain_{'i8' if layout == 'int8' else 'bits'}"
    Eo, Mo = o.sweep_series(beta, n, 0, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.sweep(beta, 2, L, 1); o.sweep(beta, 2, L, 1)
    _same_state(g, o)
    # a call of four sweeps or more: every half-sweep in one cooperative launch, the lattice on chip (k_grid_plain: every tile
    # active in every phase, two exchange records per tile used in turn)
    sfx = "i8" if layout == "int8" else "bits"
    g.sweep(beta, 5, 0, k); o.sweep(beta, 5, 0, k)
    assert g.sweep_path() == f"grid_plain_{sfx}"
    _same_state(g, o)
    g.sweep(beta, 4, L, 1); o.sweep(beta, 4, L, 1)              # again: the exchange records are reset per call
    assert g.sweep_path() == f"grid_plain_{sfx}"
    _same_state(g, o)


def test_grid_plain_kernel_several_jobs_per_warp():
    """k_grid_plain with the number of resident warps capped (ISING_GRID_WARPS, a testing aid): several register-tile jobs of
    each colour per warp, as on lattices of 2^24 sites; fresh process because the cap is read once."""
    import os, subprocess, sys
    code = (
        "import numpy as np, paper_1006_3865_b200 as P\n"
        "from oracle import oracle as O\n"
        "import ising_workloads as W\n"
        "P.use_torch()\n"
        "for (L, T, k, n, seeds, bits, jseed) in ((1024, 0, 1, 4, [5], False, None), (768, 16, 2, 2, [6, 7], True, None), (704, 8, 1, 3, [8], False, 5), (1024, 128, 1, 2, [9], True, None)):\n"
        "    J = W.couplings(2, L, jseed) if jseed is not None else None\n"
        "    g = P.Ising(2, L, coupling=J, seeds=seeds); o = O.Oracle(2, L, seeds=seeds, J=J)\n"
        "    if bits: g.set_layout(P.ISING_LAYOUT_BITS)\n"
        "    g.sweep(0.44, n, T, k); o.sweep(0.44, n, T, k)\n"
        "    assert g.sweep_path().startswith('grid_plain' if T == 0 else 'grid_masked'), g.sweep_path()\n"
        "    assert np.array_equal(np.asarray(g.copy_spins()).reshape(-1), np.asarray(o.spins()).reshape(-1))\n"
        "    Eg, Mg = g.observables(); Eo, Mo = o.observables()\n"
        "    assert list(Eg) == list(Eo) and list(Mg) == list(Mo)\n"
        "print('capped ok')\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for cap in ("24", "100"):
        out = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, ISING_GRID_WARPS=cap),
                             capture_output=True, text=True, timeout=900)
        assert out.returncode == 0 and "capped ok" in out.stdout, out.stderr[-2000:]


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,k,n,beta,seeds,jseed,path", [
    (16, 1, 4, BC3, [4], None, "resident3d_plain"),
    (32, 2, 3, BC3, [4, 5], None, "resident3d_plain"),
    (64, 1, 2, 0.3, [9], None, "resident3d_plain"),
    (32, 1, 3, 0.9, [1, 2], 7, "resident3d_plain"),        # 3D +-J
    (96, 1, 2, BC3, [2], None, "tile3d_plain"),             # L > 64: a launch per half-sweep
    (80, 2, 2, 0.9, [3], 11, "tile3d_plain"),
])
def test_plain_checkerboard_3d(P, orc, L, k, n, beta, seeds, jseed, path, layout):
    """a8 in 3D: tile == L on the 8^3 register tiling, cluster-resident (L <= 64) or a launch per half-sweep."""
    J = W.couplings(3, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 3, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(beta, n, 0, k); o.sweep(beta, n, 0, k)
    assert g.sweep_path() == f"{path}_{'i8' if layout == 'int8' else 'bits'}"
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, L, k)
    Eo, Mo = o.sweep_series(beta, n, L, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.sweep(beta, 2, 8, 1); o.sweep(beta, 2, 8, 1)          # and back to the double checkerboard
    _same_state(g, o)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds,jseed,path", [
    (64, 16, 1, 4, BC2, [3], None, "resident_masked"),       # the paper's tile sizes 4, 8, 16
    (128, 8, 2, 3, BC2, [5], None, "resident_masked"),
    (128, 4, 1, 3, 0.6, [6, 7], None, "resident_masked"),
    (64, 2, 3, 2, 0.3, [8], None, "resident_masked"),
    (256, 16, 4, 2, 1.0, [100, 101], 5, "resident_masked"),  # +-J
    (512, 128, 2, 2, BC2, [11], None, "resident_masked"),    # tiles above 64: whole register tiles switched on and off
    (1024, 256, 1, 2, 0.5, [12], None, "grid_masked"),       # beyond the cluster: on chip on all SMs (k_grid_plain) ...
    (1024, 128, 2, 1, BC2, [13], None, "grid_masked"),
    (1024, 16, 1, 2, BC2, [9], None, "grid_masked"),
    (704, 8, 2, 1, 0.5, [10, 11], None, "grid_masked"),
    (704, 4, 1, 3, 1.0, [100], 5, "grid_masked"),            # +-J
    (1024, 16, 1, 1, BC2, [9], None, "tile_masked"),         # ... unless the call is too short to pay for it: a launch per half-sweep
])
def test_small_coarse_tiles_on_the_fast_kernels(P, orc, L, tile, k, n, beta, seeds, jseed, path, layout):
    """Double checkerboard with coarse tiles smaller than a register tile: masked half-sweeps, same trajectory as the oracle's
    (the series call that follows takes a launch per half-sweep at the sizes beyond the cluster)."""
    J = W.couplings(2, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 2, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(beta, n, tile, k); o.sweep(beta, n, tile, k)
    assert g.sweep_path() == f"{path}_{'i8' if layout == 'int8' else 'bits'}"
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.sweep(beta, 2, 32, 1); o.sweep(beta, 2, 32, 1)
    _same_state(g, o)


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds,jseed,path", [
    (16, 4, 1, 4, BC3, [4], None, "resident3d_masked"),
    (32, 2, 2, 2, BC3, [5], None, "resident3d_masked"),
    (32, 16, 1, 3, 0.3, [6, 7], None, "resident3d_masked"),     # coarse tiles of 2 x 2 x 2 register tiles
    (64, 4, 1, 2, 0.9, [1, 2], 7, "resident3d_masked"),         # +-J
    (96, 4, 1, 2, BC3, [2], None, "tile3d_masked"),
    (128, 32, 2, 1, BC3, [3], None, "tile3d_masked"),
])
def test_other_coarse_tiles_3d(P, orc, L, tile, k, n, beta, seeds, jseed, path, layout):
    """3D double checkerboard with coarse tiles other than 8 on the 8^3 register tiling (masked half-sweeps)."""
    J = W.couplings(3, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 3, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.sweep(beta, n, tile, k); o.sweep(beta, n, tile, k)
    assert g.sweep_path() == f"{path}_{'i8' if layout == 'int8' else 'bits'}"
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)


GRID = [
    # L, tile, k, n, beta, seeds, jseed: more than 64 warp jobs per colour -> the grid-resident kernel (one cooperative launch)
    (1024, 32, 4, 3, BC2, [2], None),          # config 2 shape
    (1024, 64, 1, 4, BC2, [3], None),
    (768, 32, 2, 3, 0.3, [5, 6], None),        # replicas; B = 24
    (704, 32, 1, 5, BC2, [9], None),           # B = 22: 121 jobs per colour, ragged against every CTA size
    (1152, 64, 2, 2, 0.6, [8], None),          # B = 18
    (640, 32, 2, 3, 1.0, [100, 101], 5),       # +-J glass, replicas share the coupling records
    (768, 64, 1, 3, 0.8, [7], 11),
    (2048, 32, 1, 2, BC2, [3], None),          # 1024 jobs per colour
    (1024, 32, 2, 2, 0.0, [2], None),          # beta = 0: every proposal accepted
    (1024, 64, 2, 2, 30.0, [2], None),         # thresholds underflow to 0
]


@pytest.mark.parametrize("jit", ["off", "on"])
@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds,jseed", GRID)
def test_grid_resident_kernel_matches_oracle(P, orc, L, tile, k, n, beta, seeds, jseed, layout, jit):
    """512 < L <= 4096 (the paper's own sizes), n >= 2 passes: one cooperative launch, every tile on chip for the
    whole call, boundary words exchanged through versioned 64-bit words in L2 (k_grid_planes).  jit "off": at these sizes the
    producer / consumer form (one consumer warp + three producer warps per pair of jobs); jit "on": the run-time specialised
    kernel, every warp on its own.  With and without the E/M series; composing with the per-pass kernels."""
    J = W.couplings(2, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 2, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.set_jit(jit)
    sfx = "i8" if layout == "int8" else "bits"
    g.sweep(beta, n, tile, k); o.sweep(beta, n, tile, k)
    assert g.sweep_path() == f"grid_planes_{sfx}"
    assert g.last_sweep_specialized() == (jit == "on" and beta > 0)
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n + 1, tile, k)                 # E and M after every pass, counted on the registers
    assert g.sweep_path() == f"grid_planes_{sfx}"
    Eo, Mo = o.sweep_series(beta, n + 1, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.sweep(beta, 1, tile, k); o.sweep(beta, 1, tile, k)          # a single pass: the per-pass kernel, same trajectory
    assert g.sweep_path() == f"tile_planes_{sfx}"
    g.force_path(2)
    g.sweep(beta, 2, tile, k); o.sweep(beta, 2, tile, k)
    assert g.sweep_path() == f"tile_planes_{sfx}"
    _same_state(g, o)
    if len(seeds) > 1:
        assert g.overlap(0, 1) == o.overlap(0, 1)


def test_grid_resident_kernel_several_jobs_per_warp():
    """The same kernel with the number of resident warps capped (ISING_GRID_WARPS, a testing aid): 2, 4, ... jobs of each colour
    per warp, tile state parked in shared memory between phases; fresh process because the cap is read once."""
    import os, subprocess, sys
    code = (
        "import numpy as np, paper_1006_3865_b200 as P\n"
        "from oracle import oracle as O\n"
        "P.use_torch()\n"
        "for (L, T, k, n, seeds, bits) in ((1024, 32, 2, 3, [5], False), (768, 64, 1, 3, [6, 7], True), (704, 32, 1, 4, [8], False)):\n"
        "    g = P.Ising(2, L, seeds=seeds); o = O.Oracle(2, L, seeds=seeds)\n"
        "    if bits: g.set_layout(P.ISING_LAYOUT_BITS)\n"
        "    Eg, Mg = g.sweep_series(0.44, n, T, k); Eo, Mo = o.sweep_series(0.44, n, T, k)\n"
        "    assert g.sweep_path().startswith('grid_planes'), g.sweep_path()\n"
        "    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)\n"
        "    assert np.array_equal(np.asarray(g.copy_spins()).reshape(-1), np.asarray(o.spins()).reshape(-1))\n"
        "print('capped ok')\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for cap in ("40", "100"):
        out = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, ISING_GRID_WARPS=cap),
                             capture_output=True, text=True, timeout=900)
        assert out.returncode == 0 and "capped ok" in out.stdout, out.stderr[-2000:]


def test_grid_resident_kernel_run_time_build_without_parked_constants():
    """The run-time build of the same kernel in the form that holds BASELINE config 3 on chip (one CTA per SM, geometry and
    threshold heads compiled in, up to 16 jobs of a colour per warp, the jobs' constants decoded in every phase instead of
    parked in shared memory: ISING_G2_PARK=0, a testing aid, forces that form on lattices the oracle finishes in seconds),
    with and without the E / M series (two different builds), replicas (per-replica Philox keys) and +-J couplings.  Where the
    jobs per warp divide the jobs of a tile row, tile 32 runs as strips (left / right neighbours from the warp's own shared
    memory, ISING_G2_STRIP in grid_planes_device.cuh): caps 64 and 128 at L = 1024 (4 and 2 jobs per warp; 8 and 4 with two
    replicas), cap 24 at L = 640 (a whole tile row per warp: the strip's ends are each other's neighbours)."""
    import os, subprocess, sys
    code = (
        "import numpy as np, paper_1006_3865_b200 as P\n"
        "from oracle import oracle as O\n"
        "import ising_workloads as W\n"
        "P.use_torch()\n"
        "for (L, T, k, n, seeds, bits, jseed, beta) in ((1024, 32, 1, 4, [5], False, None, 0.4406868), (768, 64, 2, 3, [6, 7], True, None, 0.44),\n"
        "                                              (640, 32, 1, 3, [8], False, 5, 1.0), (1024, 64, 1, 5, [9], False, None, 0.4406868),\n"
        "                                              (1024, 32, 2, 3, [10, 11], True, None, 0.5),\n"
        "                                              (832, 32, 1, 3, [12], True, 5, 1.0)):\n"     # 13 tiles of a colour per row: jobs straddle rows, no strips
        "    J = W.couplings(2, L, jseed) if jseed is not None else None\n"
        "    g = P.Ising(2, L, coupling=J, seeds=seeds); o = O.Oracle(2, L, seeds=seeds, J=J)\n"
        "    g.set_jit('on')\n"
        "    if bits: g.set_layout(P.ISING_LAYOUT_BITS)\n"
        "    g.sweep(beta, n, T, k); o.sweep(beta, n, T, k)\n"
        "    assert g.sweep_path().startswith('grid_planes') and g.last_sweep_specialized(), g.sweep_path()\n"
        "    assert np.array_equal(np.asarray(g.copy_spins()).reshape(-1), np.asarray(o.spins()).reshape(-1))\n"
        "    Eg, Mg = g.sweep_series(beta, n, T, k); Eo, Mo = o.sweep_series(beta, n, T, k)\n"
        "    assert g.sweep_path().startswith('grid_planes') and g.last_sweep_specialized(), g.sweep_path()\n"
        "    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)\n"
        "    assert np.array_equal(np.asarray(g.copy_spins()).reshape(-1), np.asarray(o.spins()).reshape(-1))\n"
        "print('unparked ok')\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for cap in ("24", "64", "128"):
        out = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, ISING_GRID_WARPS=cap, ISING_G2_PARK="0"),
                             capture_output=True, text=True, timeout=900)
        assert out.returncode == 0 and "unparked ok" in out.stdout, out.stderr[-2000:]


@pytest.mark.parametrize("dim,L,tile,k,rng,layout,R,jseed", [
    (2, 128, 32, 2, "planes", "int8", 5, 5),       # plane records, 0/1 bytes
    (2, 128, 64, 1, "planes", "bits", 16, 7),      # bit records, two pair chunks per row (R - 1 > 8)
    (2, 64, 32, 1, "planes", "int8", 2, None),
    (3, 16, 8, 2, "planes", "int8", 4, 3),         # 3D records
    (3, 32, 8, 1, "planes", "bits", 3, None),
    (2, 128, 32, 1, "words", "int8", 4, None),     # row-major tile records: through the canonical array
    (2, 36, 6, 1, "planes", "int8", 3, None),      # generic kernels: canonical array
    (2, 64, 0, 2, "planes", "int8", 3, None),      # 64 x 64 plain checkerboard
])
def test_overlap_all_matches_oracle(P, orc, dim, L, tile, k, rng, layout, R, jseed):
    """ising_overlap_all: every Q_ab in one call, computed where the spins live (XOR + popcount on the records), against the
    oracle's pairwise definition; before the first sweep (canonical array), after sweeps, and again after a read-only call."""
    J = W.couplings(dim, L, jseed) if jseed is not None else None
    seeds = [300 + 7 * r for r in range(R)]
    g, o = _both(P, orc, dim, L, seeds, J, rng)
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)

    def want():
        Q = np.zeros((R, R), dtype=np.int64)
        for a in range(R):
            for b in range(R):
                Q[a, b] = o.overlap(a, b)
        return Q
    assert np.array_equal(g.overlap_all(), want())
    g.sweep(0.7, 3, tile, k); o.sweep(0.7, 3, tile, k)
    Q = want()
    assert np.array_equal(np.diag(Q), np.full(R, L ** dim))
    assert np.array_equal(g.overlap_all(), Q)
    s = np.asarray(g.copy_spins()).reshape(R, -1)              # a read-only call converts the records once ...
    assert np.array_equal(s, np.asarray(o.spins()).reshape(R, -1))
    assert np.array_equal(g.overlap_all(), Q) and g.overlap(0, R - 1) == Q[0, R - 1]
    g.sweep(0.7, 1, tile, k); o.sweep(0.7, 1, tile, k)         # ... and a sweep invalidates that copy
    assert np.array_equal(np.asarray(g.copy_spins()).reshape(R, -1), np.asarray(o.spins()).reshape(R, -1))
    import torch
    Qd = torch.zeros((R, R), dtype=torch.int64, device="cuda")
    g.overlap_all(Qd)
    assert np.array_equal(Qd.cpu().numpy(), want())


GRID3 = [
    # L, k, n, beta, seeds, jseed: more than 64 warp jobs per colour -> k_grid3d (one cooperative launch)
    (80, 1, 3, BC3, [4], None),              # B = 10
    (96, 2, 2, BC3, [5], None),              # B = 12
    (128, 1, 3, BC3, [9], None),             # 2^21 sites
    (80, 1, 3, 0.3, [5, 6], None),           # replicas
    (96, 1, 2, 0.9, [2], 10),                # 3D Edwards-Anderson glass
    (80, 2, 2, 0.0, [2], None),
    (80, 2, 2, 9.0, [2], None),
]


@pytest.mark.parametrize("jit", ["off", "on"])
@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,k,n,beta,seeds,jseed", GRID3)
def test_grid_resident_3d_kernel_matches_oracle(P, orc, L, k, n, beta, seeds, jseed, layout, jit):
    """3D lattices beyond the cluster (L > 64; BASELINE config 4 is L = 256): the whole call in one cooperative launch,
    slices on chip, the six faces of every tile exchanged as versioned 64-bit words in L2 (k_grid3d)."""
    J = W.couplings(3, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 3, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.set_jit(jit)
    sfx = "i8" if layout == "int8" else "bits"
    g.sweep(beta, n, 8, k); o.sweep(beta, n, 8, k)
    assert g.sweep_path() == f"grid3d_planes_{sfx}"
    assert g.last_sweep_specialized() == (jit == "on" and beta > 0 and jseed is None)
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, 8, k)
    assert g.sweep_path() == f"grid3d_planes_{sfx}"
    Eo, Mo = o.sweep_series(beta, n, 8, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.sweep(beta, 1, 8, k); o.sweep(beta, 1, 8, k)                # a single pass: the per-pass kernel
    assert g.sweep_path() == f"tile3d_planes_{sfx}"
    _same_state(g, o)


def test_grid_resident_3d_kernel_several_jobs_per_warp():
    """k_grid3d with the number of resident warps capped (ISING_GRID_WARPS): several jobs of each colour per warp."""
    import os, subprocess, sys
    code = (
        "import numpy as np, paper_1006_3865_b200 as P\n"
        "from oracle import oracle as O\n"
        "P.use_torch()\n"
        "for (L, k, n, seeds, bits) in ((80, 2, 3, [5], False), (96, 1, 3, [6, 7], True)):\n"
        "    g = P.Ising(3, L, seeds=seeds); o = O.Oracle(3, L, seeds=seeds)\n"
        "    if bits: g.set_layout(P.ISING_LAYOUT_BITS)\n"
        "    Eg, Mg = g.sweep_series(0.2216546, n, 8, k); Eo, Mo = o.sweep_series(0.2216546, n, 8, k)\n"
        "    assert g.sweep_path().startswith('grid3d_planes'), g.sweep_path()\n"
        "    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)\n"
        "    assert np.array_equal(np.asarray(g.copy_spins()).reshape(-1), np.asarray(o.spins()).reshape(-1))\n"
        "print('capped ok')\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, ISING_GRID_WARPS="50"),
                         capture_output=True, text=True, timeout=900)
    assert out.returncode == 0 and "capped ok" in out.stdout, out.stderr[-2000:]


FLOW = [
    # L, tile, k, n, beta, seeds, jseed
    (256, 32, 1, 3, BC2, [3], None),
    (256, 64, 2, 3, BC2, [4], None),
    (384, 32, 1, 5, 0.3, [5, 6], None),        # replicas; B = 12: tile rows of 3 two-slot jobs
    (192, 32, 2, 4, 1.0, [7], 5),              # B = 6: one slot per lane (B/2 odd); +-J
    (320, 64, 1, 6, BC2, [8], None),           # B = 5 is odd: not a valid double checkerboard -> skipped below
    (1024, 64, 1, 4, BC2, [8], None),
    (2048, 32, 1, 3, BC2, [9], None),
    (256, 32, 1, 2, 0.0, [2], None),
    (256, 64, 1, 2, 30.0, [2], None),
]


@pytest.mark.parametrize("jit", ["off", "on"])
@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("L,tile,k,n,beta,seeds,jseed", [c for c in FLOW if (c[0] // c[1]) % 2 == 0])
def test_data_flow_kernel_matches_oracle(P, orc, L, tile, k, n, beta, seeds, jseed, layout, jit):
    """k_flow_planes: all passes of a call in ONE persistent launch, the coarse colours ordered by per-tile progress counters
    instead of kernel boundaries (the path bench.py times at L = 16384, k = 1).  force_path(4) keeps the on-chip kernels
    out of the way so that small lattices reach it; then the per-pass kernels continue the same trajectory."""
    J = W.couplings(2, L, jseed) if jseed is not None else None
    g, o = _both(P, orc, 2, L, seeds, J, rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.set_jit(jit)
    g.force_path(4)
    sfx = "i8" if layout == "int8" else "bits"
    g.sweep(beta, n, tile, k); o.sweep(beta, n, tile, k)
    assert g.sweep_path() == f"flow_planes_{sfx}"
    assert g.last_sweep_specialized() == (jit == "on" and beta > 0)
    _same_state(g, o)
    g.sweep(beta, n + 1, tile, k); o.sweep(beta, n + 1, tile, k)      # again: scratch counters are reset per call
    _same_state(g, o)
    g.force_path(3)                                                   # no data-flow kernel: a launch per colour
    g.sweep(beta, 2, tile, k); o.sweep(beta, 2, tile, k)
    assert g.sweep_path() in (f"tile_planes_{sfx}", f"resident_planes_{sfx}", f"grid_planes_{sfx}")
    _same_state(g, o)


@pytest.mark.parametrize("dim,L,tile,k,n,beta,R", [
    (2, 64, 32, 1, 3, 1.0, 33), (2, 128, 32, 2, 2, 0.8, 64), (2, 128, 64, 1, 2, 1.2, 48), (2, 128, 32, 2, 2, 0.0, 40),   # several word lattices
    (2, 64, 32, 1, 2, 1.0, 100),
    (3, 16, 8, 1, 3, 0.9, 8), (3, 32, 8, 2, 2, 0.5, 32), (3, 16, 8, 2, 2, 1.1, 50), (3, 48, 8, 1, 2, 0.9, 5),            # 3D: the EA glass of P:100
    (3, 16, 8, 1, 2, 0.0, 3), (3, 16, 8, 1, 2, 9.0, 64),
])
def test_multi_realisation_batch_wide_and_3d(P, orc, dim, L, tile, k, n, beta, R):
    """Asynchronous multi-spin coding beyond the first slice ("missing" 6): more than 32 realisations per handle
    (several 32-bit word lattices driven by the same random numbers), and the 3D Edwards-Anderson glass (8^3 tiles); every
    realisation against the oracle's multi batch."""
    Js = np.stack([W.couplings(dim, L, 700 + r) for r in range(R)])
    seeds = [3000 + r for r in range(R)]
    g = P.Ising(dim, L, coupling=Js, seeds=seeds, sweep_seed=777)
    o = orc.Oracle(dim, L, J=Js, seeds=seeds, sweep_seed=777, rng="words")
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, n, tile, k)
    assert g.sweep_path() == "amsc"
    Eo, Mo = o.sweep_series(beta, n, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.sweep(beta, 2, tile, k); o.sweep(beta, 2, tile, k)
    _same_state(g, o)
    assert g.overlap(0, R - 1) == o.overlap(0, R - 1)
    Q = g.overlap_all()
    assert Q[1, R - 1] == o.overlap(1, R - 1) and Q[0, 0] == L ** dim
