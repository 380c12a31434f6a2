import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle_lib():
    from oracle import projector
    projector.lib()
    return projector


def pytest_addoption(parser):
    parser.addoption("--shim-as-cuda", action="store_true", default=False,
                     help="TEST TOOLING: run the gpu-marked tests WITHOUT a GPU, the kernel sources under tests/cpu_shim standing in "
                          "for the device (tests/fake_cuda.py).  Checks the tests' own host logic; claims nothing about the device.")


@pytest.fixture(scope="session", autouse=True)
def _shim_as_cuda(request):
    if not request.config.getoption("--shim-as-cuda"):
        yield
        return
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    from fake_cuda import shim_as_cuda
    with shim_as_cuda():
        yield
