import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "timing: wall-clock evidence (cost-model fits); never part of the gpu parity gate")


@pytest.fixture(scope="session")
def oracle():
    """The CPU oracle (built with gcc on first use)."""
    from oracle import lpo
    lpo.lib()
    return lpo


def read_golden(name):
    """Rows of a tests/golden/*.txt fixture: '#' lines are citations/comments."""
    path = os.path.join(ROOT, "tests", "golden", name)
    rows = []
    with open(path) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows
