"""GPU parity at the full sizes of BASELINE.json's five configs, through the C ABI, in the launch
configuration bench.py times.  Expected values (E, M, FNV-1a-64 of the canonical spins at given
passes; for config 2 also hashes of the whole E and M series) come from

  * tests/golden/survey_appendix_a.json — SURVEY.md Appendix A, RNG mapping "words"
    (two unrelated scratch programs of the survey), and
  * tests/golden/oracle_goldens.json — written by tests/golden/make_goldens.py, which calls only
    oracle/, RNG mapping "planes" (the library default).

No expected value comes from the CUDA path.  Integer work: the bar is exact equality."""
import json
import os

import numpy as np
import pytest

import ising_workloads as W

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))
SURVEY = json.load(open(os.path.join(HERE, "golden", "survey_appendix_a.json")))
_OG = os.path.join(HERE, "golden", "oracle_goldens.json")
ORACLE = json.load(open(_OG)) if os.path.exists(_OG) else {}


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1006_3865_b200 as pkg
    pkg.use_torch()
    return pkg


def _state(g, orc, R):
    s = np.asarray(g.copy_spins()).reshape(R, -1)
    E, M = g.observables()
    return [int(v) for v in E], [int(v) for v in M], ["%016x" % orc.hash_bytes(s[r]) for r in range(R)]


@pytest.mark.parametrize("case", SURVEY["cases"], ids=lambda c: c["name"])
def test_survey_appendix_a_words(P, orc, case):
    """Every Appendix A trajectory, full length, RNG mapping words."""
    J = W.couplings(case["dim"], case["L"], case["jseed"]) if case.get("jseed") is not None else None
    g = P.Ising(case["dim"], case["L"], coupling=J, seed=case["seed"], rng="words")
    done = 0
    for p, E, M, h in case["checkpoints"]:
        g.sweep(case["beta"], p - done, case["tile"], case["k"])
        done = p
        Eg, Mg, hg = _state(g, orc, 1)
        assert (Eg[0], Mg[0], hg[0]) == (E, M, h), f"{case['name']} pass {p} ({g.sweep_path()})"
    g.destroy()


PLANES_JOBS = ["c2_beta0.3", "c2_beta0.4", "c2_beta0.4406868", "c2_beta0.5", "c2_beta0.6"] + \
    [f"c3_L{L}_t{T}_k{k}" for L in (16384, 2048) for T in (32, 64) for k in (1, 4, 16)] + \
    ["c3_L16384_plain", "c4_plain", "c4_k1", "c4_k4", "c5_all16", "c5_seed100", "c5_seed101", "c5_seed114", "c5_seed115"]


@pytest.mark.parametrize("layout", ["int8", "bits"])
@pytest.mark.parametrize("name", PLANES_JOBS)
def test_oracle_goldens_planes(P, orc, name, layout):
    """Configs 2-5 at full size, RNG mapping planes, both HBM layouts, against stored oracle runs."""
    if name not in ORACLE:
        pytest.skip(f"{name} not in oracle_goldens.json (run tests/golden/make_goldens.py)")
    job = ORACLE[name]
    assert job.get("rng", "planes") == "planes"
    R = len(job["seeds"])
    J = W.couplings(job["dim"], job["L"], job["jseed"]) if "jseed" in job else None
    g = P.Ising(job["dim"], job["L"], coupling=J, seeds=job["seeds"], rng="planes")
    if layout == "bits":
        g.set_layout(P.ISING_LAYOUT_BITS)
    done = 0
    Es, Ms = [], []
    for cp in job["checkpoints"]:
        p = cp[0]
        if p > done:
            if job.get("series"):
                E, M = g.sweep_series(job["beta"], p - done, job["tile"], job["k"])
                Es.append(np.asarray(E)); Ms.append(np.asarray(M))
            else:
                g.sweep(job["beta"], p - done, job["tile"], job["k"])
            done = p
        Eg, Mg, hg = _state(g, orc, R)
        assert (Eg, Mg, hg) == (cp[1], cp[2], cp[3]), f"{name} pass {p} ({g.sweep_path()})"
        extra = cp[4:]
        if job.get("series") and p > 0:
            assert "%016x" % orc.hash_bytes(np.ascontiguousarray(np.concatenate(Es)).astype("<i8")) == extra[0]
            assert "%016x" % orc.hash_bytes(np.ascontiguousarray(np.concatenate(Ms)).astype("<i8")) == extra[1]
            extra = extra[2:]
        if job.get("overlaps") and p > 0:                 # config 5's declared output: all 120 pairwise overlaps, one call
            Q = g.overlap_all()
            for key, q in extra[0].items():
                a, b = (int(v) for v in key.split(","))
                assert Q[a, b] == q and Q[b, a] == q
            assert g.overlap(0, R - 1) == extra[0][f"0,{R - 1}"]
    if job["dim"] == 2 and job["tile"] in (32, 64) and job["L"] > 64:
        sfx = "i8" if layout == "int8" else "bits"
        assert g.sweep_path() in (f"tile_planes_{sfx}", f"resident_planes_{sfx}", f"grid_planes_{sfx}")
    if job["tile"] == job["L"]:
        assert g.sweep_path() == ("tile_plain_" if job["dim"] == 2 else "tile3d_plain_") + ("i8" if layout == "int8" else "bits")
    elif job["dim"] == 3:
        sfx = "i8" if layout == "int8" else "bits"
        assert g.sweep_path() in (f"tile3d_planes_{sfx}", f"resident3d_planes_{sfx}", f"grid3d_planes_{sfx}")
    g.destroy()


def test_config1_planes_series_against_live_oracle(P, orc):
    """Config 1 in full (L=64, plain checkerboard, 1000 sweeps, E and M after every sweep): the oracle finishes it
    in seconds, so it is run live."""
    c = W.CONFIGS[1]
    g = P.Ising(2, c["L"], seed=c["seed"], rng="planes")
    o = orc.Oracle(2, c["L"], seed=c["seed"], rng="planes")
    Eg, Mg = g.sweep_series(c["beta"], c["n"], c["tile"], c["k"])
    Eo, Mo = o.sweep_series(c["beta"], c["n"], c["tile"], c["k"])
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)
    assert np.array_equal(np.asarray(g.copy_spins()), o.spins())
    assert g.sweep_path() == "plain64_planes_i8"
