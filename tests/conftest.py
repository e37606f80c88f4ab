import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def orc():
    """Long-double CPU oracle (the parity truth)."""
    from oracle.binding import Oracle
    return Oracle("ld")


@pytest.fixture(scope="session")
def orc_d():
    """fp64 instantiation of the same oracle source (the fp64 rounding floor)."""
    from oracle.binding import Oracle
    return Oracle("d")
