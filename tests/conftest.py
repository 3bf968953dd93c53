import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running parity case")


def golden(name):
    """Rows of a whitespace-separated fixture under tests/golden/ (lines starting with # are citations)."""
    rows = []
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


@pytest.fixture(scope="session")
def water_oracle():
    import oracle
    from paper_1503_01722_b200 import workloads as W
    cfg = W.config(1)
    return oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
