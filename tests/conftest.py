"""pytest configuration: registers the `gpu` marker.

`-m "not gpu"` runs here on CPU (oracle pins, host logic, C-ABI symbol export, gloo);
`-m gpu` runs on a B200 and goes through the C-ABI library only.
"""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle():
    from oracle import lofar_oracle
    lofar_oracle.build()
    return lofar_oracle
