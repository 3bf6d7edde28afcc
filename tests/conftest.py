import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "codegen: runs with the NVRTC-specialised contraction kernel enabled")


@pytest.fixture(scope="session")
def lib():
    """The C-ABI binding; GPU tests fail loudly if the extension is missing."""
    import paper_2510_00193_b200 as m
    return m


@pytest.fixture(autouse=True)
def _codegen_off_unless_asked(request, monkeypatch):
    """NVRTC specialisation of the contraction kernel costs seconds per potential: GPU tests run the interpreted
    kernel (bit-identical by construction and by test) unless they are marked `codegen`."""
    if request.node.get_closest_marker("codegen") is None:
        monkeypatch.setenv("MTP_TREE_CODEGEN", "0")
    else:
        monkeypatch.delenv("MTP_TREE_CODEGEN", raising=False)
