import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: full BASELINE.json sizes")


def read_golden(name):
    """key = value text fixtures; '#' starts a comment.  Values parsed as float (fractions 'p/q' allowed)."""
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = (t.strip() for t in line.split("=", 1))
            if "/" in v:
                p, q = v.split("/")
                out[k] = float(p) / float(q)
            else:
                out[k] = float(v)
    return out


@pytest.fixture(scope="session")
def golden():
    return read_golden
