import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "huge: full-size L=65536 oracle transition check (opt-in: SW_RUN_HUGE=1)")


GOLDEN = os.path.join(ROOT, "tests", "golden")


def read_golden(name):
    """Lines of a golden fixture without comments and blanks."""
    out = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                out.append(line)
    return out


@pytest.fixture(scope="session")
def golden():
    return read_golden
