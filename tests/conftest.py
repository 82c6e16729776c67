import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg0():
    import synth
    return synth.config0()


@pytest.fixture(scope="session")
def cfg0_cal(cfg0):
    import oracle
    return oracle.calibrate_frame(cfg0)


@pytest.fixture(scope="session")
def cfg0_fp(cfg0):
    import oracle
    idx, dmin = oracle.footprint(cfg0.wcs, cfg0.shape[1], cfg0.shape[0], cfg0.nside)
    return idx, dmin
