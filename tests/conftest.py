import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (runs on the B200 box only)")


@pytest.fixture(scope="session")
def ref():
    """The CPU oracle (oracle/ref.py); builds oracle/libjdft_ref.so on first use."""
    from oracle import ref as _ref
    _ref.lib()
    return _ref


def _have_cuda():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


@pytest.fixture(scope="session")
def jd():
    """The CUDA binding (paper_1708_03621_b200.binding).  GPU tests only; fails loudly if the library is missing."""
    if not _have_cuda():
        pytest.skip("no CUDA device")
    import paper_1708_03621_b200.binding as binding
    return binding
