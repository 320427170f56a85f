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


def _library_path():
    return os.path.join(ROOT, "paper_1605_07023_b200", "libgridb200.so")


def pytest_collection_modifyitems(config, items):
    """The CUDA library is built in-tree (git-ignored).  Only the tests that load it need it: the -m gpu tests and
    tests/test_boundary_cpu.py (which builds it through its own fixture).  The oracle's pins and the multi-rank
    test run on any host, with or without nvcc; if a checkout has no library and it cannot be built, the tests
    that need it fail loudly on importing the binding (no skip, no fallback) -- nothing else is affected."""
    needs = [it for it in items if it.get_closest_marker("gpu") is not None]
    if not needs or os.path.exists(_library_path()):
        return
    try:
        import __graft_entry__ as entry
        entry.build()
    except Exception as exc:                                   # noqa: BLE001
        # no skip: each of those tests then fails loudly on importing the binding ("libgridb200.so is missing")
        print(f"conftest: libgridb200.so is missing and could not be built here: {exc}", file=sys.stderr)
