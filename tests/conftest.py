import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: exhaustive full-size runs (minutes of CPU oracle time); need FT_RUN_SLOW=1")


@pytest.fixture(scope="session")
def golden():
    """tests/golden/closed_forms.txt: name value  # citation"""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", "closed_forms.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                name, val = line.split()
                out[name] = float(val)
    return out
