import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run on the GPU box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    """GPU tests must FAIL (not skip) on a GPU box without the extension; on a CPU box
    they are deselected by -m "not gpu".  Nothing to do here beyond registering."""
    return


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.lib()
    return oracle
