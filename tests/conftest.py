import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: long-running full-size parity case (skipped unless QW_RUN_SLOW=1)")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("QW_RUN_SLOW") == "1":
        return
    skip = pytest.mark.skip(reason="slow full-size case: set QW_RUN_SLOW=1")
    for item in items:
        if "slow" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session")
def oracle():
    import oracle as _oracle

    _oracle.build()
    return _oracle


@pytest.fixture(scope="session")
def qw():
    """The ctypes binding over libqw.so (built on demand; fails loudly if nvcc is missing)."""
    from paper_1003_3779_b200 import binding, build

    build.build()
    binding.load()
    return binding
