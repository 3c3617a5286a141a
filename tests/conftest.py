import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_addoption(parser):
    parser.addoption("--slow", action="store_true", default=False, help="also run the tests marked slow (mutation check)")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")
    config.addinivalue_line("markers", "slow: minutes of CPU time; skipped unless --slow is given")


def pytest_collection_modifyitems(config, items):
    if config.getoption("--slow"):
        return
    skip = pytest.mark.skip(reason="slow: run with --slow")
    for item in items:
        if "slow" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session")
def cfg0():
    import tpcsynth
    return tpcsynth.generate(0)


@pytest.fixture(scope="session")
def cfg1_small():
    """Config-1 kinematics at 1500 tracks (36 sectors): seconds for the oracle."""
    import tpcsynth
    return tpcsynth.generate(1, n_tracks=1500)
