import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def emo():
    """The oracle binding (builds oracle/libemo.so with gcc on first use)."""
    from oracle import emo as m
    m.lib()
    return m


def golden(name):
    """Read a tests/golden/*.txt fixture: '#' comments, whitespace-separated columns."""
    rows = []
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows
