import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a real B200 (run with -m gpu on the GPU box)")


@pytest.fixture(scope="session")
def ref():
    """The oracle binding (oracle/ref.py); builds oracle/liblrmd_ref.so on first use."""
    from oracle import ref as _ref
    _ref.max_threads()
    return _ref


@pytest.fixture(scope="session")
def lrmd():
    """The CUDA path's binding (paper_1212_0262_b200/lrmd.py); builds/loads liblrmd.so.
    GPU tests fail (not skip) when the library or the device is missing: no silent fallback."""
    from paper_1212_0262_b200 import lrmd as _lrmd
    _lrmd.load()
    return _lrmd


@pytest.fixture(scope="session")
def inputs():
    from paper_1212_0262_b200 import inputs as _inputs
    return _inputs
