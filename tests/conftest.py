import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """The suites need the in-tree libfresnel.so (there is no CPU fallback): compile it with nvcc if a fresh
    checkout does not have it yet.  A failed build is left for the tests to report."""
    from paper_1806_06467_b200 import binding, build
    if not os.path.exists(binding.LIB_PATH):
        try:
            build.build(verbose=True)
        except Exception as exc:      # noqa: BLE001
            print(f"could not build libfresnel.so: {exc}", file=sys.stderr)
    yield


@pytest.fixture(scope="session")
def oracle():
    from oracle import oracle as O
    O.lib()
    return O
