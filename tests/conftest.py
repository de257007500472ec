import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    # The built library is git-ignored: (re)build it in-tree when it is missing or stale, so that a
    # fresh checkout can run the tests.  The binding itself never builds or falls back.
    import importlib.util
    spec = importlib.util.spec_from_file_location("gf_b200_build", os.path.join(ROOT, "paper_1305_3440_b200", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build()


@pytest.fixture(scope="session")
def cuda_device():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu test selected but no CUDA device is visible")
    return torch.device("cuda:0")
