import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (sm_100a); run with -m gpu on the B200 box")


def golden(name):
    """Numbers of a fixture under tests/golden/ (lines starting with # are citations/comments)."""
    vals = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, val = line.split("=", 1)
            vals[key.strip()] = val.strip()
    return vals


@pytest.fixture(scope="session")
def lib():
    """The CUDA path's Python binding; fails loudly if the extension is missing."""
    import paper_1511_03614_b200 as fb
    fb.load()
    return fb
