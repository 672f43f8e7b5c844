import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def c1():
    from paper_2112_11991_b200 import workloads
    return workloads.config1()


def pytest_terminal_summary(terminalreporter):
    """What the full-size parity tests actually compared (SURVEY 8(d) protocol), also under -q."""
    try:
        from parity import SUMMARY
    except ImportError:
        return
    if SUMMARY:
        terminalreporter.section("parity sample")
        for line in SUMMARY:
            terminalreporter.write_line(line)
