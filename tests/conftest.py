import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")


@pytest.fixture(scope="session")
def oracle():
    """The float64 CPU oracle (built with gcc on first use)."""
    import oracle as _oracle

    _oracle.build()
    return _oracle


@pytest.fixture(scope="session")
def cobalt():
    """The CUDA library binding; fails loudly when the extension is missing."""
    import paper_1801_04834_b200 as pkg

    pkg.load()
    return pkg
