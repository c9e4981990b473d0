import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")


def pytest_collection_modifyitems(config, items):
    """GPU tests fail loudly (not skip) when selected without a device; they are deselected on
    the CPU box with -m "not gpu"."""
    return


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


@pytest.fixture
def set_debug():
    """dash_hash4d_set_debug(key, value) for one test; every touched key is reset to 0 (library default) after."""
    import paper_2507_19141_b200 as dh
    used = []

    def _set(key, value):
        dh.dash_hash4d_set_debug(key, value)
        used.append(key)

    yield _set
    for key in used:
        dh.dash_hash4d_set_debug(key, 0)
