import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: long-running parity case")


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """libcp4d.so is built in-tree (nvcc cross-compiles without a GPU); a no-op when it is up to date."""
    from paper_1809_09725_b200 import build
    build.build_lib()


@pytest.fixture(scope="session")
def oracle():
    from oracle import ref
    ref.build()
    ref.set_threads(1)
    return ref
