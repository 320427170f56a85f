import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """The CUDA library is built in-tree (git-ignored): build it if this checkout has none yet."""
    import __graft_entry__ as entry
    if not os.path.exists(os.path.join(ROOT, "paper_1605_07023_b200", "libgridb200.so")):
        entry.build()
