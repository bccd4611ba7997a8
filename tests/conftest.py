import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def read_golden(name):
    """Parse a tests/golden/*.txt fixture: 'key | value | citation' lines, '#' comments."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, val, _cite = [s.strip() for s in line.split("|", 2)]
            out[key] = val
    return out


@pytest.fixture(scope="session")
def oracle():
    from oracle import nbs_oracle
    return nbs_oracle
