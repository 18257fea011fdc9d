import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running full-size case")


@pytest.fixture(scope="session")
def oracle_lib():
    """Build (if stale) and load the CPU oracle."""
    from oracle import build_oracle
    return build_oracle.build()


@pytest.fixture(autouse=True)
def _workspace_guard(request):
    """After every GPU test: no context bound with poison=True wrote past the end of its workspace."""
    yield
    if request.node.get_closest_marker("gpu") is None:
        return
    from paper_1803_03498_b200 import binding
    for g in list(binding.POISONED):
        assert g.workspace_guard_intact(), "a kernel or copy wrote past heom_workspace_bytes()"
