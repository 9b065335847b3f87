import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def tiny_local():
    """configs[0] with adjacent probes (duplicates occur), on the CPU."""
    from workloads import CONFIGS, make_workload
    return make_workload(CONFIGS["tiny_local"])


@pytest.fixture(scope="session")
def tiny():
    from workloads import CONFIGS, make_workload
    return make_workload(CONFIGS["tiny"])
