import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def kho():
    """The CPU oracle binding (test infrastructure)."""
    from oracle import kho as _kho
    _kho.lib()
    return _kho


def read_golden():
    """tests/golden/paper_values.txt -> {name: value}: the numbers PAPER.md prints (each with its citation in the file)."""
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) == 2:
                vals[line[0]] = float(line[1])
    return vals


@pytest.fixture(scope="session")
def golden():
    return read_golden()
