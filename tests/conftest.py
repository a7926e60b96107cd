import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a B200 (run with -m gpu on the GPU box)")
    config.addinivalue_line("markers", "slow: long-running check, off by default (NB_SLOW=1)")


def pytest_collection_modifyitems(config, items):
    if os.environ.get("NB_SLOW") == "1":
        return
    skip = pytest.mark.skip(reason="set NB_SLOW=1 to run")
    for it in items:
        if "slow" in it.keywords:
            it.add_marker(skip)


@pytest.fixture(scope="session", autouse=True)
def _fresh_library_on_a_gpu_box(request):
    """On a box with a GPU the library is rebuilt from the sources of this tree before the first
    test, so that what the GPU tests load is what the tree says (the shipped .so is a convenience)."""
    try:
        import torch
        have_gpu = torch.cuda.is_available()
    except ImportError:
        have_gpu = False
    if have_gpu and os.environ.get("NB_NO_REBUILD") != "1":
        import __graft_entry__ as g
        g.build(force=True)
    yield
