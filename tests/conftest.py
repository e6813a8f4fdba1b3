import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu on the GPU box)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import fe_oracle
    fe_oracle.lib()
    return fe_oracle


@pytest.fixture(scope="session")
def fe():
    """The CUDA path's Python binding.  Fails loudly if the extension is missing or no B200 is present."""
    from paper_1412_8754_b200 import fe as _fe
    _fe.lib()
    return _fe
