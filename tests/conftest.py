import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_modifyitems(config, items):
    """GPU tests must never pass by silently skipping: on a box without CUDA they are deselected
    by `-m "not gpu"`; if selected anyway they fail loudly in the binding (no CPU fallback)."""
    return


@pytest.fixture(scope="session")
def oracle():
    from oracle import oracle as O

    O.build()
    return O
