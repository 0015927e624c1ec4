import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: full-size configs (R2B8/R2B9); still part of -m gpu")


GOLDEN = os.path.join(ROOT, "tests", "golden")


def read_golden(name):
    """rows of whitespace-split tokens, comments (#) and blank lines dropped"""
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


_grid_cache = {}


@pytest.fixture(scope="session")
def oracle_grid(oracle_mod):
    def get(k, seed=0, flags=0):
        key = (k, seed, flags)
        if key not in _grid_cache:
            _grid_cache[key] = oracle_mod.Grid(k, seed, flags)
        return _grid_cache[key]
    return get
