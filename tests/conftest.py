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
    from oracle import gf_oracle
    gf_oracle.build()
    return gf_oracle


@pytest.fixture(scope="session", autouse=True)
def _libgf_built():
    """The in-tree libgf.so is a build artefact (git-ignored): make sure it exists and is up to date before any
    test imports the binding (nvcc cross-compiles without a GPU; a no-op when nothing changed)."""
    from paper_1212_5221_b200 import build
    build.build()
