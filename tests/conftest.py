import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: full-length check against the oracle (minutes of host time); run with -m \"gpu and slow\" or RFIM_RUN_SLOW=1")


def pytest_collection_modifyitems(config, items):
    """Full-length runs stay out of the default selections (`-m gpu`, `-m "not gpu"`): they need ~20 minutes of oracle time."""
    if "slow" in (config.getoption("-m") or "") or os.environ.get("RFIM_RUN_SLOW"):
        return
    skip = pytest.mark.skip(reason='full-length run: select with -m "gpu and slow" or set RFIM_RUN_SLOW=1')
    for item in items:
        if "slow" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.lib()
    return oracle
