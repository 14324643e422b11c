import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    """Every GPU test gets a time limit (pytest-timeout, if it is installed): the one-launch-per-call kernels wait for their
    neighbours' data, and a kernel that waits for ever must fail its test, not hold the GPU box until somebody kills the job."""
    if not config.pluginmanager.hasplugin("timeout"):
        return
    for item in items:
        if "gpu" in item.keywords and item.get_closest_marker("timeout") is None:
            item.add_marker(pytest.mark.timeout(1500, method="thread"))


@pytest.fixture(scope="session")
def orc():
    """The sequential CPU oracle (test infrastructure)."""
    from oracle import oracle as O
    O.build()
    return O


@pytest.fixture(params=["planes", "words"])
def both_rngs(request, orc):
    """Run the test body under both RNG->site mappings of the oracle (DESIGN.md §3 R6)."""
    old = orc.DEFAULT_RNG
    orc.DEFAULT_RNG = request.param
    yield request.param
    orc.DEFAULT_RNG = old
