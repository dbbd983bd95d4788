import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle():
    """The CPU fp64 oracle (test infrastructure).  Built on first use with gcc."""
    import oracle as _oracle

    _oracle.build()
    return _oracle


@pytest.fixture(scope="session")
def fbp():
    """The CUDA binding.  GPU tests must run the native library: no fallback, fail loudly."""
    import torch

    import paper_2109_02174_b200 as pkg

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    pkg.load_library()  # raises if libfbp.so is missing
    return pkg
