"""GPU parity at the edges of the key and counter space, and at full length ("What's missing" 2).

* "seed: 64-bit Philox key" — every kernel family with seeds whose high word is not zero
  (k1 = seed >> 32 in every kernel);
* the random of site i in half-sweep H = 2t + c carries lo32(H), hi32(H) in the counter —
  every kernel family swept across t = 2^31 (hi32(H) goes 0 -> 1) and at t = 2^40 + 5;
* "int8-vs-bits GPU hashes must agree at full length" — the six config-3 trajectories, all 200 passes
  at L = 16384, both layouts (and the pre-compiled against the run-time specialised kernel on one of them).

All against the live oracle except the full-length run, which compares the two HBM layouts with each other
(the oracle pins the first two passes at this size and all 200 at L = 2048: test_gpu_configs.py)."""
import numpy as np
import pytest

import ising_workloads as W

pytestmark = pytest.mark.gpu

BC2, BC3 = W.BETA_C_2D, W.BETA_C_3D
WIDE_SEEDS = [(1 << 40) + 13, 0xFEDCBA9876543210]
COUNTERS = [(1 << 31) - 2, (1 << 40) + 5]


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1006_3865_b200 as pkg
    pkg.use_torch()
    return pkg


def _same_state(g, o):
    sg = np.asarray(g.copy_spins()).reshape(-1)
    so = np.asarray(o.spins()).reshape(-1)
    bad = np.flatnonzero(sg != so)
    assert bad.size == 0, f"{bad.size} spins differ, first at {bad[:8]} ({g.sweep_path()})"
    Eg, Mg = g.observables()
    Eo, Mo = o.observables()
    assert list(Eg) == list(Eo) and list(Mg) == list(Mo)


# kernel family: dim, L, tile, k, n, beta, jseed, rng, layout, force_path, jit, expected path prefix
FAMILIES = {
    "tile_planes_t32_i8": (2, 256, 32, 2, 4, BC2, None, "planes", "int8", 2, "off", "tile_planes_i8"),
    "tile_planes_t64_bits": (2, 256, 64, 1, 4, BC2, None, "planes", "bits", 2, "off", "tile_planes_bits"),
    "tile_planes_t64_i8_jit": (2, 256, 64, 2, 4, BC2, None, "planes", "int8", 2, "on", "tile_planes_i8"),
    "tile_planes_t32_bits_jit": (2, 192, 32, 1, 4, 0.3, None, "planes", "bits", 2, "on", "tile_planes_bits"),
    "tile_planes_pmj": (2, 128, 32, 4, 4, 1.0, 5, "planes", "int8", 2, "off", "tile_planes_i8"),
    "tile_planes_pmj_jit": (2, 128, 64, 2, 4, 1.0, 5, "planes", "bits", 2, "on", "tile_planes_bits"),
    "resident_planes": (2, 256, 32, 2, 4, BC2, None, "planes", "int8", 0, "auto", "resident_planes_i8"),
    "resident_planes_pmj": (2, 128, 64, 1, 4, 0.8, 11, "planes", "bits", 0, "auto", "resident_planes_bits"),
    "resident_plain": (2, 128, 0, 2, 4, BC2, None, "planes", "int8", 0, "auto", "resident_plain_i8"),
    "resident_masked": (2, 128, 8, 1, 4, BC2, None, "planes", "int8", 0, "auto", "resident_masked_i8"),
    "grid_planes": (2, 768, 32, 2, 4, BC2, None, "planes", "int8", 0, "off", "grid_planes_i8"),
    "grid_planes_jit": (2, 768, 64, 1, 4, BC2, None, "planes", "bits", 0, "on", "grid_planes_bits"),
    "grid_planes_pmj": (2, 640, 32, 1, 4, 1.0, 5, "planes", "int8", 0, "auto", "grid_planes_i8"),
    "grid3d": (3, 80, 8, 1, 4, BC3, None, "planes", "int8", 0, "off", "grid3d_planes_i8"),
    "grid3d_jit": (3, 80, 8, 2, 4, BC3, None, "planes", "bits", 0, "on", "grid3d_planes_bits"),
    "plain64": (2, 64, 0, 1, 6, BC2, None, "planes", "int8", 0, "auto", "plain64_planes_i8"),
    "tile_plain": (2, 704, 0, 1, 4, BC2, None, "planes", "int8", 2, "auto", "tile_plain_i8"),
    "tile_masked": (2, 704, 16, 1, 4, BC2, None, "planes", "bits", 2, "auto", "tile_masked_bits"),
    "grid_plain": (2, 704, 0, 1, 4, BC2, None, "planes", "int8", 0, "auto", "grid_plain_i8"),
    "grid_masked": (2, 704, 16, 1, 4, BC2, None, "planes", "bits", 0, "auto", "grid_masked_bits"),
    "grid_masked_pmj": (2, 704, 8, 2, 2, 1.0, 5, "planes", "int8", 0, "auto", "grid_masked_i8"),
    "tile3d": (3, 32, 8, 2, 4, BC3, None, "planes", "int8", 2, "off", "tile3d_planes_i8"),
    "tile3d_jit": (3, 32, 8, 1, 4, BC3, None, "planes", "bits", 2, "on", "tile3d_planes_bits"),
    "tile3d_pmj": (3, 32, 8, 1, 4, 0.9, 7, "planes", "int8", 2, "off", "tile3d_planes_i8"),
    "resident3d": (3, 32, 8, 2, 4, BC3, None, "planes", "int8", 0, "auto", "resident3d_planes_i8"),
    "resident3d_plain": (3, 32, 0, 1, 4, BC3, None, "planes", "bits", 0, "auto", "resident3d_plain_bits"),
    "tile3d_plain": (3, 96, 0, 1, 4, BC3, None, "planes", "int8", 0, "auto", "tile3d_plain_i8"),
    "tile_i8_words": (2, 128, 32, 2, 4, BC2, None, "words", "int8", 0, "auto", "tile_i8"),
    "generic_words": (2, 36, 6, 2, 4, BC2, None, "words", "int8", 1, "auto", "generic"),
    "generic_planes_3d": (3, 12, 6, 1, 4, BC3, None, "planes", "int8", 1, "auto", "generic"),
}


def _run_family(P, orc, fam, seed, t0):
    dim, L, tile, k, n, beta, jseed, rng, layout, force, jit, path = FAMILIES[fam]
    J = W.couplings(dim, L, jseed) if jseed is not None else None
    seeds = [seed, seed ^ 0x5555555500000001]
    g = P.Ising(dim, L, coupling=J, seeds=seeds, rng=rng)
    o = orc.Oracle(dim, L, seeds=seeds, J=J, rng=rng)
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    g.force_path(force)
    g.set_jit(jit)
    _same_state(g, o)                                   # the hot start uses the whole 64-bit key too (S8c.3)
    g.counter = t0; o.counter = t0
    g.sweep(beta, n, tile, k); o.sweep(beta, n, tile, k)
    assert g.sweep_path().startswith(path), g.sweep_path()
    if jit == "on":
        assert g.last_sweep_specialized()
    assert g.counter == o.counter == t0 + n * k
    _same_state(g, o)
    Eg, Mg = g.sweep_series(beta, 2, tile, k)           # the series variants of the same kernels
    Eo, Mo = o.sweep_series(beta, 2, tile, k)
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)
    g.destroy()


@pytest.mark.parametrize("seed", WIDE_SEEDS, ids=["seed_2p40_13", "seed_fedcba98"])
@pytest.mark.parametrize("fam", list(FAMILIES))
def test_seed_with_high_word(P, orc, fam, seed):
    """k1 = seed >> 32 != 0 in every kernel family."""
    _run_family(P, orc, fam, seed, 0)


@pytest.mark.parametrize("t0", COUNTERS, ids=["t_2p31_m2", "t_2p40_5"])
@pytest.mark.parametrize("fam", list(FAMILIES))
def test_counter_past_32_bits(P, orc, fam, t0):
    """hi32(H) != 0, H = 2t + c: t = 2^31 - 2 crosses the carry inside the call, t = 2^40 + 5 starts beyond it."""
    _run_family(P, orc, fam, 77, t0)


@pytest.mark.parametrize("what", ["seed", "counter_lo", "counter_hi"])
def test_amsc_wide_key_and_counter(P, orc, what):
    """The asynchronous multi-spin kernel (R17): wide sweep key and init keys, counters past 32 bits."""
    L, R, T, k, n, beta = 128, 8, 32, 2, 3, 1.0
    Js = np.stack([W.couplings(2, L, 900 + r) for r in range(R)])
    wide = what == "seed"
    seeds = [((0xABCDEF01 << 32) if wide else 0) + 2000 + r for r in range(R)]
    sweep_seed = 0xFEDCBA9876543210 if wide else 4242
    g = P.Ising(2, L, coupling=Js, seeds=seeds, sweep_seed=sweep_seed)
    o = orc.Oracle(2, L, J=Js, seeds=seeds, sweep_seed=sweep_seed, rng="words")
    _same_state(g, o)
    t0 = {"seed": 0, "counter_lo": COUNTERS[0], "counter_hi": COUNTERS[1]}[what]
    g.counter = t0; o.counter = t0
    Eg, Mg = g.sweep_series(beta, n, T, k)
    Eo, Mo = o.sweep_series(beta, n, T, k)
    assert g.sweep_path() == "amsc"
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    _same_state(g, o)


@pytest.mark.parametrize("what", ["seed0", "seed1", "counter_lo", "counter_hi"])
@pytest.mark.parametrize("dim,L,T,k,path", [(2, 64, 32, 2, "heis_tile"), (3, 16, 8, 1, "heis_tile"), (2, 20, 10, 1, "heis_generic")])
def test_heisenberg_wide_key_and_counter(P, what, dim, L, T, k, path):
    """The continuous-spin path (include/heisenberg.h): same key and counter edges, spins bit for bit."""
    from oracle import heisenberg as HO
    seed = {"seed0": WIDE_SEEDS[0], "seed1": WIDE_SEEDS[1]}.get(what, 6)
    t0 = {"counter_lo": COUNTERS[0], "counter_hi": COUNTERS[1]}.get(what, 0)
    g = P.Heisenberg(dim, L, seed=seed); o = HO.HeisenbergOracle(dim, L, seed=seed)
    g.counter = t0; o.counter = t0
    g.sweep(0.7, 4, T, k); o.sweep(0.7, 4, T, k)
    assert g.sweep_path() == path
    assert g.counter == o.counter == t0 + 4 * k
    sg = np.asarray(g.copy_spins()).view(np.uint32).reshape(3, -1)
    assert np.array_equal(sg, o.spins().view(np.uint32))


@pytest.mark.parametrize("k", [1, 4, 16])
@pytest.mark.parametrize("tile", [32, 64])
def test_config3_full_length_int8_equals_bits(P, orc, tile, k):
    """BASELINE config 3 in full: L = 16384, 200 passes, the launch configuration bench.py times (run-time specialised
    kernel), int8 records against bit records: identical canonical spins (compared on the device), E and M; the first
    two passes of every trajectory are the oracle's (tests/golden/oracle_goldens.json)."""
    import json
    import os
    import torch
    L, n = 16384, 200
    gold = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_goldens.json")))
    cps = {cp[0]: cp for cp in gold[f"c3_L16384_t{tile}_k{k}"]["checkpoints"]}
    a = P.Ising(2, L, seed=3); b = P.Ising(2, L, seed=3)
    b.set_layout(P.ISING_LAYOUT_BITS)
    sa = torch.empty(L * L, dtype=torch.int8, device="cuda")
    sb = torch.empty(L * L, dtype=torch.int8, device="cuda")
    done = 0
    for p in (2, 50, n):
        n_call = p - done
        a.sweep(BC2, n_call, tile, k); b.sweep(BC2, n_call, tile, k)
        done = p
        # int8 records at k = 1: the whole lattice on chip (a call of 8 passes or more), else the persistent data-flow
        # kernel; k > 1 and bit records: a launch per colour
        # (launch_grid_one's rule, measured: on chip up to k = 3, at tile 32 for int8 records only)
        want = "tile_planes_i8" if k > 1 else ("grid_planes_i8" if n_call >= 8 else "flow_planes_i8")
        want_b = "grid_planes_bits" if (k == 1 and tile == 64 and n_call >= 8) else "tile_planes_bits"
        assert a.sweep_path() == want and b.sweep_path() == want_b
        assert a.last_sweep_specialized() and b.last_sweep_specialized()
        a.copy_spins(sa); b.copy_spins(sb)
        assert torch.equal(sa, sb), f"int8 and bit records differ after pass {p}"
        Ea, Ma = a.observables(); Eb, Mb = b.observables()
        assert (int(Ea[0]), int(Ma[0])) == (int(Eb[0]), int(Mb[0]))
        if p in cps:                                        # the oracle's values where it has been run
            assert [int(Ea[0])] == cps[p][1] and [int(Ma[0])] == cps[p][2]
            assert "%016x" % orc.hash_bytes(sa.cpu().numpy()) == cps[p][3][0]
    if (tile, k) == (64, 1):                                # the pre-compiled kernel walks the same 200 passes
        c = P.Ising(2, L, seed=3)
        c.set_jit("off")
        c.sweep(BC2, n, tile, k)
        assert not c.last_sweep_specialized()
        c.copy_spins(sb)
        assert torch.equal(sa, sb), "pre-compiled and run-time specialised kernels differ after 200 passes"
        c.destroy()
        d = P.Ising(2, L, seed=3)                           # ... and so do a launch per colour
        d.force_path(2)
        d.sweep(BC2, n, tile, k)
        assert d.sweep_path() == "tile_planes_i8"
        d.copy_spins(sb)
        assert torch.equal(sa, sb), "on-chip kernel and per-colour launches differ after 200 passes"
        d.destroy()
        e = P.Ising(2, L, seed=3)                           # ... and the data-flow kernel
        e.force_path(4)
        e.sweep(BC2, n, tile, k)
        assert e.sweep_path() == "flow_planes_i8"
        e.copy_spins(sb)
        assert torch.equal(sa, sb), "on-chip and data-flow kernels differ after 200 passes"
        e.destroy()
    a.destroy(); b.destroy()


@pytest.mark.parametrize("L,tile,k,jobs,layout",
                         [(L, T, k, j, lay) for (L, T, k, j) in [(4096, 32, 1, 1), (4096, 64, 2, 1), (8192, 32, 1, 4), (8192, 32, 3, 4), (8192, 64, 1, 2), (8192, 64, 3, 2)]
                          for lay in ("int8", "bits")]
                         + [(5184, 32, 1, 2, "int8"),      # 81 tiles of a colour per row: a job of two tiles may straddle rows (no strips)
                            (16384, 64, 1, 8, "int8"), (16384, 64, 2, 8, "bits"), (16384, 32, 1, 16, "int8"), (16384, 32, 3, 16, "int8")])
def test_on_chip_kernel_equals_a_launch_per_colour_at_full_size(P, L, tile, k, jobs, layout):
    """Lattices of 2^24, 2^26 and 2^28 sites (BASELINE config 3: all of the GPU's shared memory) in the launch configurations the
    library chooses for them (run-time build of k_grid_planes: `jobs` jobs of a colour per warp, from L = 8192 on without parked constants and, at tile 32, as strips): the whole
    call on chip against a launch per coarse colour (ising_force_path 2) — canonical spins compared on the device, E, M and the
    series of the on-chip call against observables of the other.  Both paths are pinned to the oracle on small lattices
    (test_gpu_parity.py); this checks the full-size geometry (147 CTAs, 28 warps each)."""
    import torch
    n = 9
    a = P.Ising(2, L, seed=12); b = P.Ising(2, L, seed=12)
    if layout == "bits":
        a.set_layout(P.ISING_LAYOUT_BITS); b.set_layout(P.ISING_LAYOUT_BITS)
    b.force_path(2)
    sfx = "i8" if layout == "int8" else "bits"
    a.sweep(BC2, n, tile, k); b.sweep(BC2, n, tile, k)
    assert a.sweep_path() == f"grid_planes_{sfx}" and a.last_sweep_specialized() and b.sweep_path() == f"tile_planes_{sfx}"
    sa = torch.empty(L * L, dtype=torch.int8, device="cuda"); sb = torch.empty_like(sa)
    a.copy_spins(sa); b.copy_spins(sb)
    assert torch.equal(sa, sb), "on-chip kernel and per-colour launches differ"
    E, M = a.sweep_series(BC2, n, tile, k)                  # the series build of the same kernel
    assert a.sweep_path() == f"grid_planes_{sfx}"
    b.sweep(BC2, n - 1, tile, k)
    Eb, Mb = b.observables()
    assert (int(E[n - 2][0]), int(M[n - 2][0])) == (int(Eb[0]), int(Mb[0]))
    b.sweep(BC2, 1, tile, k)
    a.copy_spins(sa); b.copy_spins(sb)
    assert torch.equal(sa, sb)
    Ea, Ma = a.observables(); Eb, Mb = b.observables()
    assert (int(Ea[0]), int(Ma[0])) == (int(Eb[0]), int(Mb[0])) == (int(E[n - 1][0]), int(M[n - 1][0]))
    a.destroy(); b.destroy()


@pytest.mark.parametrize("dim,L,tile", [(2, 128, 32), (2, 64, 0), (3, 16, 8), (2, 1024, 32)])
def test_thresholds_straddling_2p32(P, orc, dim, L, tile):
    """0 < beta < ~1.4e-17: exp(-4 beta) rounds to 1 (thr[1] = 2^32: always accept) while exp(-8 beta) does not
    (thr[2] = 2^32 - 1).  The multi-spin kernels fold "thr = 2^32" into one mask, so this call must take the generic
    kernels, which compare each threshold on its own; same trajectory as the oracle."""
    beta = 1e-17
    assert orc.thresholds(beta, dim)[0] == 1 << 32 and orc.thresholds(beta, dim)[1] == (1 << 32) - 1
    assert P.ising_thresholds(beta, dim) == orc.thresholds(beta, dim)
    g = P.Ising(dim, L, seed=5); o = orc.Oracle(dim, L, seed=5)
    g.sweep(beta, 2, tile, 2); o.sweep(beta, 2, tile, 2)
    assert g.sweep_path() == "generic"
    _same_state(g, o)
    g.sweep(0.4, 2, tile, 1); o.sweep(0.4, 2, tile, 1)           # and the fast kernels are back afterwards
    assert g.sweep_path() != "generic"
    _same_state(g, o)


def test_jit_cache_is_bounded_and_allocations_keep_their_owner():
    """(a) The cache of run-time specialised kernels evicts the least recently used entry (ISING_JIT_CACHE=3 here; 64 by
    default) and re-compiles on demand: a temperature scan stays correct.  (b) A block is released through the hook it was
    allocated with, whatever ising_set_device_hooks was called with in between.  Fresh process: both touch process state."""
    import os, subprocess, sys
    code = (
        "import ctypes as C, numpy as np, torch, paper_1006_3865_b200 as P\n"
        "from paper_1006_3865_b200 import binding as B\n"
        "from oracle import oracle as O\n"
        "a = P.Ising(2, 64, seed=1)\n"                       # allocated with cudaMalloc (no hooks yet)
        "P.use_torch()\n"
        "b = P.Ising(2, 64, seed=2)\n"                       # allocated through torch
        "live = len(B._live)\n"
        "a.sweep(0.4, 2, 32, 1); a.destroy()\n"              # cudaFree, not the torch hook
        "assert len(B._live) >= live - 1\n"
        "assert P.lib().ising_set_device_hooks(None, None, None) == 0\n"
        "b.sweep(0.4, 2, 32, 1); b.destroy()\n"              # the torch hook, not cudaFree
        "assert len(B._live) < live\n"
        "P.use_torch()\n"
        "g = P.Ising(2, 128, seed=5); o = O.Oracle(2, 128, seed=5)\n"
        "g.set_jit('on'); g.force_path(2)\n"
        "for beta in (0.30, 0.35, 0.40, 0.45, 0.50, 0.30, 0.55, 0.35):\n"
        "    g.sweep(beta, 2, 32, 1); o.sweep(beta, 2, 32, 1)\n"
        "    assert g.last_sweep_specialized()\n"
        "assert np.array_equal(np.asarray(g.copy_spins()), o.spins())\n"
        "print('owners and cache ok')\n")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-c", code], cwd=root, env=dict(os.environ, ISING_JIT_CACHE="3"),
                         capture_output=True, text=True, timeout=900)
    assert out.returncode == 0 and "owners and cache ok" in out.stdout, out.stderr[-3000:]
