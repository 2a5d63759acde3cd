import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with `-m gpu`)")


def load_kv(name):
    """Parse a tests/golden/*.txt fixture of `name = value` lines (# comments carry the citations)."""
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = line.split("=", 1)
            out[k.strip()] = v.strip()
    return out


@pytest.fixture(scope="session")
def kat():
    return load_kv("standards_kat.txt")


@pytest.fixture(scope="session")
def paper_pins():
    return load_kv("paper_pins.txt")


@pytest.fixture(scope="session")
def orc():
    import oracle

    oracle.lib()
    return oracle
