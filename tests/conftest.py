import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import afno_oracle
    afno_oracle.build()
    return afno_oracle


@pytest.fixture(scope="session", autouse=True)
def _cuda_library_is_built():
    """The product library is built in-tree by `python -m paper_2208_05419_b200.build` (nvcc, sm_100a); build it when
    a checkout arrives without the artefact.  There is still no fallback: if the build fails, every test that needs
    the library fails loudly."""
    from paper_2208_05419_b200 import build
    build.build()
