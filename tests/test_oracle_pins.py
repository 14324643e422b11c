"""Pins of the oracle against things other than itself (run with -m "not gpu").

Each test names the mistake it is there to catch.  P:n = PAPER.md line n; S8c = SURVEY.md §8(c).
"""
import ctypes as C
import json
import math
import os

import numpy as np
import pytest

import ising_workloads as W

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "survey_appendix_a.json")))


# ---------------------------------------------------------------- Philox (S8c.2)
def test_philox_known_answer_vectors(orc):
    """Random123 KAT vectors: wrong multiplier/key constant, swapped lanes, 9 or 11 rounds."""
    for kat in GOLD["philox_kat"]:
        ctr = [int(v, 16) for v in kat["ctr"]]
        key = [int(v, 16) for v in kat["key"]]
        out = tuple(int(v, 16) for v in kat["out"])
        assert orc.philox4x32_10(ctr, key) == out


def test_philox_matches_curand_host_generator(orc):
    """Library cross-check: cuRAND's *host* Philox4_32_10 generator (runs on the CPU).

    Measured here: its default-ordering stream for seed S is the concatenation of
    Philox(ctr={0,0,n,0}, key={lo32 S, hi32 S}) for n = 0,1,2… (the subsequence index sits in
    counter word 2), four words per counter.  Pins the key split (lo word first), the lane
    order of the output and the ctr[2] data path, through a library that is not ours.
    """
    try:
        cr = C.CDLL("libcurand.so.10")
    except OSError:
        try:
            cr = C.CDLL("/usr/local/cuda/lib64/libcurand.so.10")
        except OSError:
            pytest.skip("libcurand not present")
    gen = C.c_void_p()
    CURAND_RNG_PSEUDO_PHILOX4_32_10 = 161
    if cr.curandCreateGeneratorHost(C.byref(gen), CURAND_RNG_PSEUDO_PHILOX4_32_10) != 0:
        pytest.skip("cuRAND host generator unavailable")
    seed = int(GOLD["curand_host_check"]["seed"], 16)
    assert cr.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    n = 64
    buf = (C.c_uint32 * n)()
    assert cr.curandGenerate(gen, buf, C.c_size_t(n)) == 0
    cr.curandDestroyGenerator(gen)
    got = [int(v) for v in buf]
    assert got[:4] == [int(v, 16) for v in GOLD["curand_host_check"]["first4"]]
    key = [seed & 0xFFFFFFFF, seed >> 32]
    mine = []
    for ctr0 in range(n // 4):
        mine += list(orc.philox4x32_10([0, 0, ctr0, 0], key))
    assert got == mine


def test_input_generator_agrees_with_oracle_couplings(orc):
    """ising_workloads.couplings (numpy) vs oracle_make_couplings (C++): two separate
    implementations of the coupling recipe, plus the SURVEY A.5 hash of the L=4096 array."""
    for dim, L, js in [(2, 16, 5), (3, 8, 77), (2, 6, 2**40 + 3)]:
        a = W.couplings(dim, L, js)
        b = orc.make_couplings(dim, L, js)
        assert np.array_equal(a, b)
        assert set(np.unique(a)) <= {-1, 1}
    J = W.couplings(2, 4096, 5)
    assert "%016x" % orc.hash_bytes(J) == GOLD["config5_couplings_hash"]
    assert abs(int(J.astype(np.int64).sum())) < 5 * math.sqrt(J.size)  # p = 1/2


# ---------------------------------------------------------------- thresholds (S8c.4, eq. (2))
def test_thresholds_against_multiprecision(orc):
    """thr[m] = floor(exp(-4 m β) 2^32): wrong factor (2m, 8m), off-by-one m, 2^31 scaling."""
    import mpmath as mp
    mp.mp.dps = 60
    rng = np.random.default_rng(12345)
    betas = [0.0, 0.30, 0.40, 0.4406868, 0.50, 0.60, 0.2216546, 1.0, 5.0, 25.0] + list(rng.uniform(0, 3, 40))
    for beta in betas:
        for dim in (2, 3):
            got = orc.thresholds(beta, dim)
            assert len(got) == dim
            for m in range(1, dim + 1):
                exact = mp.e ** (-mp.mpf(beta) * 4 * m) * 2 ** 32
                fl = int(mp.floor(exact))
                # double exp is within an ulp: the floor may differ only if `exact` sits
                # within 2^-20 of an integer (it never does for the cases below)
                if min(exact - fl, fl + 1 - exact) > mp.mpf(2) ** -20:
                    assert got[m - 1] == fl, (beta, m)
                else:
                    assert abs(got[m - 1] - fl) <= 1
    assert orc.thresholds(0.0, 2) == (2 ** 32, 2 ** 32)  # β = 0: always accept (needs 64-bit compare)


def test_thresholds_match_survey_table(orc):
    for b, vals in GOLD["thresholds"].items():
        assert list(orc.thresholds(float(b), 3)) == vals


# ---------------------------------------------------------------- trajectories
def _run_case(orc, case, max_pass):
    J = None
    if "jseed" in case:
        J = W.couplings(case["dim"], case["L"], case["jseed"])
    o = orc.Oracle(case["dim"], case["L"], seed=case["seed"], J=J, rng="words")
    done = 0
    for p, E, M, h in case["checkpoints"]:
        if p > max_pass:
            break
        o.sweep(case["beta"], p - done, case["tile"], case["k"])
        done = p
        e, m = o.observables()
        assert (int(e[0]), int(m[0]), "%016x" % o.hash()) == (E, M, h), (case["name"], p)
    return o


SMALL = [c for c in GOLD["cases"] if c["L"] ** c["dim"] <= 4096]


@pytest.mark.parametrize("case", SMALL, ids=[c["name"] for c in SMALL])
def test_survey_trajectories_small(orc, case):
    """Trajectories written down by programs outside this repo: catches any deviation in the
    RNG→site map, colour order, tile order, multi-hit counter, acceptance rule, 3D, ±J."""
    o = _run_case(orc, case, 10 ** 9)
    if "final_spins" in case:
        assert "".join("+" if v > 0 else "-" for v in o.spins()) == case["final_spins"]


MEDIUM = [(c, p) for c, p in [
    (next(c for c in GOLD["cases"] if c["name"] == "A2_config2_bc"), 10),
    (next(c for c in GOLD["cases"] if c["name"] == "A2_config2_b060"), 1),
    (next(c for c in GOLD["cases"] if c["name"] == "A2_config2_plain"), 1),
    (next(c for c in GOLD["cases"] if c["name"] == "A3_L2048_t64k1"), 2),
]]


@pytest.mark.parametrize("case,max_pass", MEDIUM, ids=[c["name"] for c, _ in MEDIUM])
def test_survey_trajectories_medium(orc, case, max_pass):
    _run_case(orc, case, max_pass)


def test_survey_overlap_pass0(orc):
    """Q_ab of two hot starts sharing J (A.5): replica batching + overlap."""
    J = W.couplings(2, 4096, 5)
    o = orc.Oracle(2, 4096, seeds=[100, 101, 114, 115], J=J, rng="words")
    assert o.overlap(0, 1) == GOLD["config5_overlaps"]["100,101"]["0"]
    assert o.overlap(2, 3) == GOLD["config5_overlaps"]["114,115"]["0"]
    assert o.overlap(1, 1) == 4096 * 4096
    E, M = o.observables()
    for r, name in enumerate(["A5_config5_s100", "A5_config5_s101", "A5_config5_s114", "A5_config5_s115"]):
        cp = next(c for c in GOLD["cases"] if c["name"] == name)["checkpoints"][0]
        assert (int(E[r]), int(M[r]), "%016x" % o.hash(r)) == tuple(cp[1:])
