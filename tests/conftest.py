import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def dfe():
    """The built library's binding (builds it first if stale)."""
    from paper_2601_08077_b200.build import build_library

    build_library()
    import paper_2601_08077_b200.binding as b

    return b


@pytest.fixture(scope="session")
def gpu_ws(dfe):
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    ws = dfe.Workspace(6 << 30)
    yield ws
    ws.close()


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")
