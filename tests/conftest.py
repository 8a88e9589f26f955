import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def read_golden_kv(name):
    """'key v1 v2 ...' lines -> {key: [[floats], ...]} (repeated keys stack)."""
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, *v = line.split()
            out.setdefault(k, []).append([float(x) for x in v])
    return out


@pytest.fixture(scope="session")
def golden_dir():
    return GOLDEN


_ORACLE_RUNS = {}


def oracle_run_cached(key, w, steps=None):
    """The oracle's result for a (full-size) workload, computed once per pytest session and shared by the fp64 and fp32
    parity tests: (state after `steps`, info, flags)."""
    if key not in _ORACLE_RUNS:
        from helpers import oracle_from_workload
        o = oracle_from_workload(w, threads=0)
        flags = o.step(w.steps if steps is None else steps, w.value, w.mode)
        _ORACLE_RUNS[key] = (o.get_state(), o.info(), flags)
    return _ORACLE_RUNS[key]
