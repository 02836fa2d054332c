"""pytest configuration: markers and import path.

`-m "not gpu"`: oracle pins, host logic, C-ABI symbol checks (run on the CPU box).
`-m gpu`      : parity tests proper, through the C-ABI, on a B200.
"""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: long-running statistical test")


def read_golden(name):
    """Parse tests/golden/<name>: '#' comment lines carry the citation; data
    lines are 'key: value value ...'.  Returns {key: [str, ...]}."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = line.split(":", 1)
            out[k.strip()] = v.split()
    return out


@pytest.fixture(scope="session")
def golden():
    return read_golden
