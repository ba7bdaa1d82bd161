import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def geom():
    from lhcb_gen import default_geom
    return default_geom()


@pytest.fixture(scope="session")
def oracle32(geom):
    from oracle.binding import Oracle
    return Oracle(geom, "f32")


@pytest.fixture(scope="session")
def oracle64(geom):
    from oracle.binding import Oracle
    return Oracle(geom, "f64")


@pytest.fixture(scope="session")
def cfg1_events():
    from lhcb_gen import config, generate
    return generate(config(1))


@pytest.fixture(scope="session")
def cfg2_small():
    from lhcb_gen import config, generate
    return generate(config(2, 24))
