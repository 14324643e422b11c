import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


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
