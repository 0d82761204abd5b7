import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "heavy: whole configured runs that take the oracle minutes each; deselected "
                                       "unless SN_HEAVY=1")


def _have_gpu() -> bool:
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    if os.environ.get("SN_HEAVY") != "1":   # deselect (not skip): the default GPU run reports no skipped test
        heavy = [it for it in items if "heavy" in it.keywords]
        if heavy:
            config.hook.pytest_deselected(items=heavy)
            items[:] = [it for it in items if "heavy" not in it.keywords]
    if _have_gpu():
        return
    skip = pytest.mark.skip(reason="no CUDA device in this container")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session")
def built_library():
    """The tests that drive the product through libsn.so request this: it builds the library (nvcc, in-tree) if the
    checkout has none yet.  The product itself never builds or falls back: paper_1909_08354_b200.sn raises when the
    library is missing.  The oracle pins do not request it: they need gcc only."""
    from paper_1909_08354_b200 import build
    return build.build()


@pytest.fixture(autouse=True)
def _library_for_product_tests(request):
    """gpu-marked tests and the host-logic / replica tests (everything that is not an oracle pin) get the library."""
    if not request.node.module.__name__.startswith("test_oracle_pins"):
        request.getfixturevalue("built_library")
    yield
