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
    from oracle import lf_oracle
    lf_oracle.build()
    return lf_oracle


@pytest.fixture(scope="session")
def geometry():
    from paper_2402_14670_b200 import datagen
    return datagen.toy_geometry()


@pytest.fixture(scope="session")
def params():
    from paper_2402_14670_b200 import datagen
    return datagen.default_params()
