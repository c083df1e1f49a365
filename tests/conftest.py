"""pytest configuration: registers the `gpu` marker and builds the CPU oracle once.

`-m "not gpu"` tests run on a GPU-less box (oracle pins, host logic, ABI symbol checks);
`-m gpu` tests are the CUDA-vs-oracle parity tests and call through the C-ABI.
"""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session", autouse=True)
def _oracle_built():
    import oracle
    oracle.build()
    oracle.set_threads(1)          # tiny lattices: no OpenMP overhead; big tests raise it
    yield
