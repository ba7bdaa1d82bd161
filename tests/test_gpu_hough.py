"""Parity of lhcb_seeding with the Hough-cluster UV seeding (reading A20) against the
oracle with orc_set_uv_hough: identical seed sets, bit-identical parameters, in both launch configurations;
and the matching that follows."""
import numpy as np
import pytest

from lhcb_gen import config, generate, truth
from oracle.binding import Oracle
from tests.parity import compare_long, compare_seeds, seed_keys

pytestmark = pytest.mark.gpu


def check(ev, nominal):
    from paper_2606_14480_b200 import Context, DeviceEvents, capacities
    c = Context(capacities.with_capacities(ev.geom) if nominal else ev.geom)
    c.lhcb_set_uv_hough(True)
    dev = DeviceEvents.from_host(ev)
    s = c.lhcb_seeding(dev)
    l = c.lhcb_matching(s, dev)
    gs, gl = c.seeds_to_host(s), c.long_to_host(l)
    assert (gs["status"] == 0).all() and (gl["status"] == 0).all()
    o = Oracle(ev.geom, "f32"); o.set_uv_hough(True)
    os_, om = o.reconstruct(ev)
    r = compare_seeds(os_, gs)
    assert r["n_orc"] == r["n_gpu"] == r["n_common"] and r["bit_equal"], r
    ok = dict(zip(range(os_["n"]), seed_keys(os_["event"], os_["half"], os_["hits"], os_["state"])))
    gk = dict(zip((int(x) for x in gs["slot"]), seed_keys(gs["event"], gs["half"], gs["hits"], gs["state"])))
    rl = compare_long(om, gl, ok, gk)
    assert rl["n_orc"] == rl["n_gpu"] == rl["n_common"] and rl["bit_equal"], rl
    # back to the iterative default: a different (larger) seed collection on these events
    c.lhcb_set_uv_hough(False)
    it = c.seeds_to_host(c.lhcb_seeding(dev))
    assert it["n"] != gs["n"] or not np.array_equal(it["hits"], gs["hits"])
    c.close()
    return r, gs, it


def test_hough_cfg1():
    r, _, _ = check(generate(config(1, 16)), nominal=False)
    assert r["n_common"] > 30 * 16


def test_hough_cfg2_both_launch_configurations():
    ev = generate(config(2, 96))
    r, gs, it = check(ev, nominal=False)
    check(ev, nominal=True)
    assert r["n_common"] > 100 * 96
    e_h = truth.seeding_summary(ev, gs["hits"])["efficiency"]; e_i = truth.seeding_summary(ev, it["hits"])["efficiency"]
    assert e_h > 0.93 and abs(e_h - e_i) < 0.03          # "similar tracking performance" (L204)


def test_hough_cfg4_high_occupancy():
    check(generate(config(4, 48)), nominal=False)
