import os
import sys
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: takes more than a few seconds on CPU")


def read_golden(name):
    """Rows of a tests/golden/*.txt fixture: (model, N, params dict, sector dict, E0)."""
    rows = []
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            tok = line.split()
            params = {k: float(v) for k, v in (kv.split("=") for kv in tok[2].split(","))}
            sector = {k: int(v) for k, v in (kv.split("=") for kv in tok[3].split(","))}
            rows.append((tok[0], int(tok[1]), params, sector, float(tok[4])))
    return rows
