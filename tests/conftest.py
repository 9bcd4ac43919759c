import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running (full-size configs)")


def load_golden_gammas():
    """gamma_x, gamma_y, gamma_z, gamma_t from tests/golden/gamma_degrand_rossi.txt."""
    val = {"0": 0, "1": 1, "-1": -1, "i": 1j, "-i": -1j}
    mats, rows = {}, None
    with open(os.path.join(GOLDEN, "gamma_degrand_rossi.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            if line in ("gx", "gy", "gz", "gt"):
                rows = mats.setdefault(line, [])
                continue
            rows.append([val[t] for t in line.split()])
    return [np.array(mats[k], dtype=np.complex128) for k in ("gx", "gy", "gz", "gt")]


@pytest.fixture(scope="session")
def gammas():
    return load_golden_gammas()
