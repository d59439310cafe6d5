"""pytest configuration: markers, import path, shared fixtures."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)  # `import gpu_util` (a top-level `tests` package may exist elsewhere)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def load_golden(name: str) -> dict:
    """Parse tests/golden/<name>: `key = hex` lines, `#` comments -> {key: bytes}."""
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = [t.strip() for t in line.split("=", 1)]
            out[k] = bytes.fromhex(v)
    return out


@pytest.fixture(scope="session")
def golden():
    return load_golden
