"""CPU-side checks of the C-ABI library: it builds, loads, and exports every symbol that
include/ising.h declares; host-only entry points behave; compute calls fail loudly without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    import paper_1006_3865_b200 as P
    P.lib()
    return P


def test_every_declared_symbol_is_exported(pkg):
    hdr = open(os.path.join(ROOT, "include", "ising.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(ising_[a-z_]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    assert declared == set(pkg.SYMBOLS)
    L = pkg.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_every_declared_heisenberg_symbol_is_exported(pkg):
    hdr = open(os.path.join(ROOT, "include", "heisenberg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(heis_[a-z_]+)\s*\(", hdr))
    assert declared and declared == set(pkg.HEIS_SYMBOLS)
    L = pkg.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert not L.heis_create(1, 8, 0) and not L.heis_create(2, 7, 0) and not L.heis_create(3, 2048, 0)
    assert L.heis_sweep(None, 0.5, 1, 0, 1) < 0 and L.heis_observables(None, None, None) < 0


def test_thresholds_host_table_matches_oracle(pkg, orc):
    # S8c.4: both sides call the host exp(); the tables must be identical
    for beta in (0.0, 0.30, 0.40, 0.4406868, 0.50, 0.60, 1.0, 0.2216546, 3.0, 7.0):
        for dim in (2, 3):
            assert pkg.ising_thresholds(beta, dim) == orc.thresholds(beta, dim)
    with pytest.raises(pkg.IsingError):
        pkg.ising_thresholds(-1.0, 2)
    with pytest.raises(pkg.IsingError):
        pkg.ising_thresholds(0.5, 4)


def test_no_cpu_fallback(pkg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(pkg.IsingError, match="no CUDA device|CPU path"):
        pkg.Ising(2, 64, seed=1)
    with pytest.raises(pkg.IsingError):
        pkg.use_torch()


def test_argument_errors_before_any_device_work(pkg):
    L = pkg.lib()
    seeds = np.array([1], dtype=np.uint64)
    for dim, Ls in ((1, 8), (4, 8), (2, 7), (2, 0), (3, 2048)):
        assert not L.ising_create_batch(dim, Ls, None, seeds.ctypes.data, 1)
        assert L.ising_last_error()
    assert L.ising_sweep(None, 0.4, 1, 0, 1) < 0
    assert L.ising_observables(None, None, None) < 0
    assert L.ising_copy_spins(None, None) < 0


def test_product_does_not_reference_the_oracle():
    """The product path may not import, include, link or execute anything under oracle/."""
    pk = os.path.join(ROOT, "paper_1006_3865_b200")
    pat = re.compile(r"(import\s+oracle|from\s+oracle|from\s+\.\.?oracle|#include\s+\"[^\"]*oracle|liboracle|oracle\.py|ising_oracle)")
    for dp, _, fs in os.walk(pk):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dp, f)).read()), f
