import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_sessionstart(session):
    # a checkout has no build artefacts (*.so are git-ignored): compile the CUDA library once, as __graft_entry__.build() does
    try:
        from paper_2307_03452_b200 import build as _b

        _b.ensure_built()
    except Exception as e:  # the ABI tests then fail loudly on the missing library
        print(f"conftest: could not build libmd4.so: {e}", file=sys.stderr)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: longer CPU test")


@pytest.fixture(scope="session")
def gpu_available():
    import torch

    return torch.cuda.is_available()
