import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

if os.path.dirname(os.path.abspath(__file__)) not in sys.path:
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def read_golden(name):
    """Rows of a tests/golden/*.txt fixture: '#' lines are citations, the rest are
    whitespace-separated fields (numbers parsed as float)."""
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            rows.append([float(x) if _isnum(x) else x for x in line.split()])
    return rows


def _isnum(s):
    try:
        float(s)
        return True
    except ValueError:
        return False


@pytest.fixture(scope="session")
def golden():
    return read_golden
