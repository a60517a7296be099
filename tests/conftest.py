import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cuda_device():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    # the in-tree libraries travel with the repository snapshot; (re)build whatever is missing or stale on this box
    from paper_2502_20610_b200 import build
    build.build()
    from oracle import build_oracle
    build_oracle.build()
    return torch.device("cuda:0")
