"""The seeded input generator: determinism, layout invariants, config shapes."""
import numpy as np

from lhcb_gen import config, generate, slice_events


def test_deterministic_and_prefix_stable():
    a = generate(config(2, 8)); b = generate(config(2, 8)); c = generate(config(2, 5))
    assert np.array_equal(a.hit_x, b.hit_x) and np.array_equal(a.ut_x0, b.ut_x0)
    # same chunk -> same first events regardless of n_events? chunks are seeded per (seed, chunk),
    # but a chunk's content depends on its size, so only full chunks are prefix-stable
    assert c.n_events == 5 and a.n_events == 8


def test_layout_invariants():
    ev = generate(config(2, 6))
    assert ev.zone_off.dtype == np.uint32 and len(ev.zone_off) == 6 * 24 + 1
    assert ev.zone_off[-1] == ev.n_hits and ev.hit_x.dtype == np.float32
    for z in range(6 * 24):
        seg = ev.hit_x[ev.zone_off[z]:ev.zone_off[z + 1]]
        assert (np.diff(seg) >= 0).all() and (np.abs(seg) < 3300).all()
    for z in range(6 * 4):
        seg = ev.ut_x0[ev.ut_off[z]:ev.ut_off[z + 1]]
        assert (np.diff(seg) >= 0).all()
    assert set(np.unique(ev.polarity)) == {-1, 1}
    assert (ev.ut_yhi - ev.ut_ylo == 100).all()
    n_per_ev = ev.n_hits / ev.n_events
    assert 3000 < n_per_ev < 4600
    # truth ids index the particle table
    assert ev.hit_pid.max() < len(ev.particles["p"]) and ev.velo_pid.min() >= 0


def test_cfg1_shape():
    ev = generate(config(1))
    assert ev.n_events == 16 and len(ev.particles["p"]) == 16 * 40 and len(ev.ut_x0) == 0
    assert (ev.hit_pid >= 0).all() and (ev.polarity == -1).all()
    assert 2000 <= ev.particles["p"].min() and ev.particles["p"].max() <= 100000


def test_cfg4_cfg5_shape():
    ev = generate(config(4, 4))
    P = ev.particles
    assert 0.1 < (P["kind"] == 2).mean() < 0.3 and P["p"].min() >= 1500
    s2 = P["tx0"] ** 2 + P["ty"] ** 2
    pt = P["p"] * np.sqrt(s2 / (1 + s2))
    assert (pt >= 200 * (1 - 1e-9))[P["p"] < 99999].all()
    ev5 = generate(config(5, 4))
    assert ev5.n_hits == 0 and ev5.seed_state.shape[0] == 5
    assert 200 < ev5.seed_state.shape[1] / 4 < 300 and 300 < len(ev5.velo_x) / 4 < 400
    assert 0.6 < (ev5.seed_pid >= 0).mean() < 0.8


def test_slice_events():
    ev = generate(config(2, 6))
    s = slice_events(ev, 2, 5)
    assert s.n_events == 3 and s.zone_off[0] == 0 and s.zone_off[-1] == s.n_hits
    assert np.array_equal(s.hit_x, ev.hit_x[ev.zone_off[48]:ev.zone_off[120]])
    assert len(s.velo_x) == s.velo_off[-1] and len(s.ut_x0) == s.ut_off[-1]
