import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def gco():
    from oracle import gco as _g
    _g.build()
    return _g


@pytest.fixture(scope="session")
def gc():
    """The CUDA path through the C ABI (fails loudly if the extension is missing)."""
    from paper_1901_06798_b200 import binding
    return binding
