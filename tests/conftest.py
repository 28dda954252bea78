import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


@pytest.fixture(autouse=True)
def _parity_context(request):
    """Names the running test in the parity helpers' margin / failure records and flushes the margins afterwards."""
    try:
        from tests import parity
    except Exception:            # CPU-only collection without torch.cuda is fine: parity is only used by gpu tests
        yield
        return
    parity.CONTEXT["test"] = request.node.name
    parity.MARGINS.clear()
    yield
    if parity.MARGINS:
        parity.dump_margins()
