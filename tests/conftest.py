import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: further exhaustive oracle pins (variant-bit x spec combinations beyond the default set); "
                                       "run with `-m slow`; the recorded pass is profiles/r3_slow_pins.txt")


def pytest_collection_modifyitems(config, items):
    """`slow` tests run only when asked for by name (-m slow / -m \"slow and not gpu\")."""
    if "slow" in (config.getoption("-m") or ""):
        return
    skip = pytest.mark.skip(reason="slow exhaustive pin: run with -m slow")
    for item in items:
        if "slow" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.build()
    return oracle
