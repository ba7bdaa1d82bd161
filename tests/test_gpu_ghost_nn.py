"""Parity of lhcb_matching with the ghost-killing network set (reading A14b) against
oracle.matching(nn=...): identical long-track sets and bit-identical ghost probabilities (both sides spell
out exp/log with the same single-rounded operations)."""
import numpy as np
import pytest

from lhcb_gen import config, generate, ghost_nn
from tests.parity import compare_long, seed_keys

pytestmark = pytest.mark.gpu


def run_both(ev, oracle32, caps=None, n_direct=False):
    from paper_2606_14480_b200 import Context, DeviceEvents, capacities
    w = ghost_nn()
    geom = capacities.with_capacities(ev.geom) if caps else ev.geom
    c = Context(geom)
    c.lhcb_set_ghost_nn(w)
    dev = DeviceEvents.from_host(ev)
    if n_direct:
        seeds, slot = c.seeds_from_states(ev.n_events, ev.seed_off, ev.seed_state)
        gl = c.long_to_host(c.lhcb_matching(seeds, dev, use_ut=True))
        om = oracle32.matching(ev.n_events, ev.seed_off, ev.seed_state.T, ev, use_ut=True, nn=w)
        ok = {i: i for i in range(ev.seed_state.shape[1])}
        gk = {int(s): i for i, s in enumerate(slot)}
    else:
        s = c.lhcb_seeding(dev)
        gl = c.long_to_host(c.lhcb_matching(s, dev, use_ut=True))
        gs = c.seeds_to_host(s)
        os_ = oracle32.seeding(ev)
        seed_off = np.zeros(ev.n_events + 1, np.uint32)
        np.cumsum(np.bincount(os_["event"], minlength=ev.n_events), out=seed_off[1:])
        om = oracle32.matching(ev.n_events, seed_off, os_["state"], ev, use_ut=True, nn=w,
                               nhits=(os_["nx"] + os_["nuv"]).astype(np.uint8))
        ok = dict(zip(range(os_["n"]), seed_keys(os_["event"], os_["half"], os_["hits"], os_["state"])))
        gk = dict(zip((int(x) for x in gs["slot"]), seed_keys(gs["event"], gs["half"], gs["hits"], gs["state"])))
    assert (gl["status"] == 0).all()
    rl = compare_long(om, gl, ok, gk)
    assert rl["n_orc"] == rl["n_gpu"] == rl["n_common"] and rl["bit_equal"], rl
    # ghost probabilities, track by track
    a, b = rl["pairs"]
    assert np.array_equal(om["ghost"][a].astype(np.float32).view(np.uint32), gl["ghost"][b].view(np.uint32))
    # switching the network off restores the chi2 ranking (A14)
    c.lhcb_set_ghost_nn(None)
    c.close()
    return om, rl


def test_nn_selection_cfg2(oracle32):
    om, rl = run_both(generate(config(2, 96)), oracle32)
    assert rl["n_common"] > 60 * 96 and (om["ghost"] < 0.8).all()


def test_nn_selection_cfg2_nominal_launch_configuration(oracle32):
    run_both(generate(config(2, 64)), oracle32, caps=True)


def test_nn_selection_cfg4(oracle32):
    run_both(generate(config(4, 48)), oracle32)


def test_nn_selection_cfg5_direct_seeds(oracle32):
    om, rl = run_both(generate(config(5, 60)), oracle32, n_direct=True)
    assert rl["n_common"] > 50 * 60
