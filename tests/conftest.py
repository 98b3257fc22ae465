import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# Lines a test wants printed after the run, pass or fail (the parity record of the full-size
# configs: E_rho / E_u per config; pytest -q hides a passing test's own prints).
RECORD_LINES = []


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: the longest GPU cases (minutes; part of the default -m gpu run)")


@pytest.fixture
def record():
    """record(line): print the line in the terminal summary."""
    return RECORD_LINES.append


def pytest_terminal_summary(terminalreporter):
    if RECORD_LINES:
        terminalreporter.write_sep("-", "parity record (GPU vs oracle)")
        for line in RECORD_LINES:
            terminalreporter.write_line(line)
