import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def load_golden(name):
    """tests/golden/<name>: 'key = value  # citation' lines -> dict of floats."""
    out = {}
    for line in (ROOT / "tests" / "golden" / name).read_text().splitlines():
        line = line.split("#", 1)[0].strip()
        if not line:
            continue
        k, v = line.split("=", 1)
        out[k.strip()] = float(v)
    return out


@pytest.fixture(scope="session")
def golden_constants():
    return load_golden("constants.txt")
