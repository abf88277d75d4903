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
    from oracle import nss_oracle
    nss_oracle.build()
    return nss_oracle


@pytest.fixture(scope="session")
def wl1(oracle):
    """config 1 with data synthesised from the oracle's waveform."""
    from paper_2509_24949_b200 import inputs
    return inputs.make_data(inputs.config1(), oracle.waveform)


@pytest.fixture(scope="session")
def wl2(oracle):
    """config 2 (B = 128) with data synthesised from the oracle's waveform."""
    from paper_2509_24949_b200 import inputs
    return inputs.make_data(inputs.config2(), oracle.waveform)
