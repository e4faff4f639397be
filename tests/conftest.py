import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import shwfs_oracle
    shwfs_oracle.build()
    return shwfs_oracle


@pytest.fixture(scope="session")
def libshwfs():
    """Path of the built C-ABI library (compiled in-tree with nvcc for sm_100a if stale or missing)."""
    from paper_1408_0698_b200 import build as b
    try:
        return b.build()
    except Exception:
        if b.LIB.exists():      # no nvcc on this box: use the library that travelled with the snapshot
            return b.LIB
        raise


@pytest.fixture(scope="session")
def gpu(libshwfs):
    """(torch, binding) on a box with a CUDA device.  The -m gpu tests must never pass on a fallback: the
    binding has none, and this fixture fails (not skips) if the library cannot be loaded."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1408_0698_b200 import binding
    binding.load()
    return torch, binding
