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


# ---- the configs at their stated sizes (BASELINE.json), generated once per session and shared by the full-size
# GPU tests; the *_full fixtures add the oracle's result (iterative UV seeding, chi2 ranking, with UT)
@pytest.fixture(scope="session")
def cfg2_events():
    from lhcb_gen import config, generate
    ev = generate(config(2), workers=8)
    assert ev.n_events == 1000
    return ev


@pytest.fixture(scope="session")
def cfg2_full(cfg2_events):
    from oracle.parallel import reconstruct_parallel
    return cfg2_events, reconstruct_parallel(cfg2_events)


@pytest.fixture(scope="session")
def cfg3_events():
    from lhcb_gen import config, generate
    ev = generate(config(3), workers=8)
    assert ev.n_events == 16384
    return ev


@pytest.fixture(scope="session")
def cfg3_full(cfg3_events):
    from oracle.parallel import reconstruct_parallel
    r = reconstruct_parallel(cfg3_events)
    print("oracle on cfg3: %d processes, %.1f s wall, %.1f core-seconds" % (r[2]["workers"], r[2]["wall_s"], r[2]["cpu_s"]))
    return cfg3_events, r


@pytest.fixture(scope="session")
def cfg4_events():
    from lhcb_gen import config, generate
    ev = generate(config(4), workers=8)
    assert ev.n_events == 2000
    return ev


@pytest.fixture(scope="session")
def cfg5_events():
    from lhcb_gen import config, generate
    ev = generate(config(5), workers=8)
    assert ev.n_events == 1000
    return ev
