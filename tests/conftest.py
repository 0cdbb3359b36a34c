import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def read_pins(name="lattice_pins.txt"):
    """tests/golden/<name>: `key = value` lines, '#' comments."""
    pins = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as fh:
        for line in fh:
            line = line.strip()
            if line and not line.startswith("#"):
                k, v = line.split("=")
                pins[k.strip()] = float(v)
    return pins


@pytest.fixture(scope="session")
def pins():
    return read_pins()
