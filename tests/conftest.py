import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    import oracle as orc

    orc.build()
    return orc


@pytest.fixture(scope="session", autouse=True)
def built_library():
    """Every test goes through libconserve_kv.so: build it (incrementally, nvcc for sm_100a) if it is missing or stale,
    so that a fresh checkout without the git-ignored .so still runs the CUDA path instead of failing to load it."""
    from paper_2606_01839_b200 import build as libbuild

    return libbuild.build_library()
