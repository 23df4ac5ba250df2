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
    """The CPU oracle (test infrastructure), compiled on first use."""
    from oracle import oracle as o
    o.build()
    return o


@pytest.fixture(scope="session")
def tiny(orc):
    """Config 0 data set (noise seed 0 + SNR-12 injection made with the oracle's template)."""
    import synthetic as syn
    return syn.make_dataset(syn.CONFIGS[0], orc.template)
