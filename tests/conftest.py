import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_addoption(parser):
    parser.addoption("--full-scan", action="store_true", default=False,
                     help="tests/test_gpu_full_scan.py: compare ALL projections of C3 and C4 with the oracle "
                          "(about 25 minutes of oracle time) and write gpurun_out/full_parity_*.json")
    parser.addoption("--random-cases", action="store", default="0",
                     help="tests/test_gpu_random_workloads.py: this many further random workloads against the oracle")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def workloads_cache():
    """Seeded workloads are deterministic; build each once per session."""
    from workloads import make_workload
    cache = {}

    def get(name, n_proj=None):
        key = (name, n_proj)
        if key not in cache:
            cache[key] = make_workload(name, n_proj=n_proj)
        return cache[key]
    return get
