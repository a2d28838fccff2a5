import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


_WORKLOADS = {}


@pytest.fixture(scope="session")
def workload():
    """workload(name, device='cpu') -> cached inputs.Workload."""
    from paper_2606_02916_b200 import inputs

    def get(name, device="cpu"):
        k = (name, str(device))
        if k not in _WORKLOADS:
            _WORKLOADS[k] = inputs.make_workload(name, device=device)
        return _WORKLOADS[k]

    return get
