"""Parity of the CUDA path with the f32 oracle on the same seeded events, through the C-ABI.

Bar (BASELINE.json north_star): hit-index sets bit-exact, except candidates whose deciding cut lies
within 1e-5 relative of a threshold (<= 0.1%); float parameters within 1e-4 relative, x within 5 um.
Both sides follow the same float32 operation order, so the expected result is exact equality.
"""
import numpy as np
import pytest

from lhcb_gen import config, default_geom, generate, truth
from tests.parity import compare_long, compare_seeds, seed_keys

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx(geom):
    from paper_2606_14480_b200 import Context
    c = Context(geom)
    yield c
    c.close()


def run_gpu(ctx, ev, use_ut=True):
    from paper_2606_14480_b200 import DeviceEvents
    dev = DeviceEvents.from_host(ev)
    s = ctx.lhcb_seeding(dev)
    assert ctx.last_launch_count() == 1
    l = ctx.lhcb_matching(s, dev, use_ut=use_ut)
    ctx.torch.cuda.synchronize()
    return ctx.seeds_to_host(s), ctx.long_to_host(l)


def check_chain(ctx, oracle32, ev, use_ut):
    gs, gl = run_gpu(ctx, ev, use_ut)
    assert (gs["status"] == 0).all() and (gl["status"] == 0).all(), "capacity overflow"
    os_, om = oracle32.reconstruct(ev, use_ut=use_ut)
    r = compare_seeds(os_, gs)
    n_diff = len(r["only_orc"]) + len(r["only_gpu"])
    assert n_diff <= 1e-3 * r["n_orc"], r
    assert r["max_rel"] <= 1e-4 and r["max_dx"] <= 5e-3, r
    ok = dict(zip(range(os_["n"]), seed_keys(os_["event"], os_["half"], os_["hits"], os_["state"])))
    gk = dict(zip((int(s) for s in gs["slot"]), seed_keys(gs["event"], gs["half"], gs["hits"], gs["state"])))
    rl = compare_long(om, gl, ok, gk)
    assert len(rl["only_orc"]) + len(rl["only_gpu"]) <= 1e-3 * max(rl["n_orc"], 1) + n_diff, rl
    assert rl["max_rel_qop"] <= 1e-4 and rl["max_rel_chi2"] <= 1e-4, rl
    # efficiency vs generator truth agrees within 0.2%
    eo = truth.seeding_summary(ev, os_["hits"])["efficiency"]
    eg = truth.seeding_summary(ev, gs["hits"])["efficiency"]
    assert abs(eo - eg) <= 2e-3
    return r, rl


def test_cfg1_tiny(ctx, oracle32, cfg1_events):
    r, rl = check_chain(ctx, oracle32, cfg1_events, use_ut=False)
    assert r["n_orc"] == r["n_gpu"] == r["n_common"] and r["bit_equal"]
    assert rl["n_orc"] == rl["n_gpu"] == rl["n_common"] and rl["bit_equal"]


def test_cfg2_nominal(ctx, oracle32):
    ev = generate(config(2, 128))
    r, rl = check_chain(ctx, oracle32, ev, use_ut=True)
    assert r["n_common"] > 100 * 128 and rl["n_common"] > 60 * 128
    assert r["bit_equal"] and rl["bit_equal"]
    assert not r["only_orc"] and not r["only_gpu"] and not rl["only_orc"] and not rl["only_gpu"]


def test_cfg4_high_occupancy(ctx, oracle32):
    ev = generate(config(4, 64))
    r, rl = check_chain(ctx, oracle32, ev, use_ut=True)
    assert r["bit_equal"] and rl["bit_equal"]
    assert not r["only_orc"] and not r["only_gpu"]


def test_cfg5_matching_stress(ctx, oracle32):
    ev = generate(config(5, 100))
    from paper_2606_14480_b200 import DeviceEvents
    dev = DeviceEvents.from_host(ev)
    seeds, slot = ctx.seeds_from_states(ev.n_events, ev.seed_off, ev.seed_state)
    gl = ctx.long_to_host(ctx.lhcb_matching(seeds, dev, use_ut=True))
    assert (gl["status"] == 0).all()
    om = oracle32.matching(ev.n_events, ev.seed_off, ev.seed_state.T, ev, use_ut=True)
    ok = {i: i for i in range(ev.seed_state.shape[1])}
    gk = {int(s): i for i, s in enumerate(slot)}
    rl = compare_long(om, gl, ok, gk)
    assert rl["n_orc"] == rl["n_gpu"] == rl["n_common"] and rl["bit_equal"], rl
    assert rl["n_common"] > 100 * 100


def test_edge_cases(ctx, oracle32, geom):
    """Empty events, an event with hits in one half only, ragged tails, unaligned tile starts."""
    from dataclasses import replace
    ev = generate(config(2, 9))
    # empty out event 3 completely and the lower half of event 5
    zo = ev.zone_off.astype(np.int64)
    keep = np.ones(ev.n_hits, bool)
    keep[zo[3 * 24]:zo[4 * 24]] = False
    keep[zo[5 * 24 + 12]:zo[6 * 24]] = False
    sizes = np.diff(zo); sizes[3 * 24:4 * 24] = 0; sizes[5 * 24 + 12:6 * 24] = 0
    new_off = np.zeros(len(zo), np.uint32); np.cumsum(sizes, out=new_off[1:])
    ev2 = replace(ev, zone_off=new_off, hit_x=ev.hit_x[keep], hit_x64=ev.hit_x64[keep], hit_pid=ev.hit_pid[keep])
    gs, gl = run_gpu(ctx, ev2)
    os_, om = oracle32.reconstruct(ev2)
    r = compare_seeds(os_, gs)
    assert r["n_orc"] == r["n_gpu"] == r["n_common"] and r["bit_equal"]
    assert not (gs["event"] == 3).any() and not ((gs["event"] == 5) & (gs["half"] == 1)).any()
    # zero events: a no-op
    from paper_2606_14480_b200 import DeviceEvents
    ev0 = generate(config(1, 1))
    dev = DeviceEvents.from_host(ev0)
    dev.n_events = 0
    ctx.lhcb_seeding(dev)
    assert ctx.last_launch_count() == 0


def test_overflow_is_reported_not_silent(geom):
    from paper_2606_14480_b200 import Context, DeviceEvents
    small = default_geom(max_seeds_per_half=16, max_xz_cand_per_half=64, max_triplets_per_half=4096)
    c = Context(small)
    ev = generate(config(2, 4))
    s = c.seeds_to_host(c.lhcb_seeding(DeviceEvents.from_host(ev)))
    assert (s["status"] & 6).any()            # candidate and/or seed overflow bits
    assert (np.bincount(s["event"] * 2 + s["half"]) <= 16).all()
    c.close()
    tiny = default_geom(max_hits_per_half=512)
    c = Context(tiny)
    s = c.seeds_to_host(c.lhcb_seeding(DeviceEvents.from_host(ev)))
    assert (s["status"] == 8).all() and s["n"] == 0
    c.close()


def test_cfg3_full_size_bench_configuration(oracle32):
    """BASELINE.json configs[2] at full size (16,384 events, seed 2) in the launch configuration bench.py
    times (capacities.NOMINAL: 256-thread seeding CTAs, 128-thread matching CTAs): no capacity overflow
    anywhere, and the events of a sample spread over the batch are identical to the oracle's, one by one."""
    from lhcb_gen import slice_events
    from paper_2606_14480_b200 import Context, DeviceEvents, capacities
    n = 16384
    ev = generate(config(3, n), workers=8)
    c = Context(capacities.with_capacities(ev.geom))
    cfgl = c.lhcb_launch_config()
    assert cfgl["seed_threads"] == 256 and cfgl["match_threads"] == 128
    gs, gl = run_gpu(c, ev, True)
    assert (gs["status"] == 0).all() and (gl["status"] == 0).all(), "capacity overflow at nominal occupancy"
    # properties that hold at any size, on the whole batch
    zo = ev.zone_off.astype(np.int64)
    hits = gs["hits"].astype(np.int64)
    zbase = (gs["event"].astype(np.int64) * 2 + gs["half"]) * 12
    for l in range(12):                                   # every hit of a seed lies in its own half's zone of that layer
        h = hits[:, l]; has = h != 0xFFFFFFFF
        assert ((h >= zo[zbase + l]) & (h < zo[zbase + l + 1]))[has].all()
    nx = (hits[:, [0, 3, 4, 7, 8, 11]] != 0xFFFFFFFF).sum(1); nuv = (hits[:, [1, 2, 5, 6, 9, 10]] != 0xFFFFFFFF).sum(1)
    assert np.array_equal(nx, gs["nx"]) and np.array_equal(nuv, gs["nuv"])
    assert np.isin(nx, (5, 6)).all() and np.isin(nuv, (4, 5, 6)).all()              # L90, A9
    assert (gs["par"][:, 5] <= 8.0).all() and (gs["par"][:, 6] <= 8.0).all()        # chi2 cuts (A6)
    assert len({(int(e), int(h)) + tuple(r) for e, h, r in zip(gs["event"], gs["half"], hits.tolist())}) == gs["n"]
    assert (gl["chi2"] < 2.0).all() and (gl["n_ut"] >= 3).all()                     # L301, L311
    assert len(np.unique(gl["seed"])) == gl["n"] and len(np.unique(gl["velo"])) == gl["n"]   # one-to-one (A14)
    vo = ev.velo_off.astype(np.int64)
    assert ((gl["velo"] >= vo[gl["event"]]) & (gl["velo"] < vo[gl["event"] + 1])).all()
    ms, ml = c.max_seeds, c.max_long
    assert (gl["seed"] // (2 * ms) == gl["event"]).all()                             # a long track's seed is of its event
    sample = [0, 1, 63, 64, 1023, 4097, 8191, 12345, 16320, 16383] + list(range(5000, 5022))
    n_s = n_l = 0
    for e in sample:
        sub = slice_events(ev, e, e + 1)
        os_, om = oracle32.reconstruct(sub, use_ut=True)
        sel = gs["event"] == e
        g1 = {k: (v[sel] if isinstance(v, np.ndarray) and v.shape[:1] == sel.shape else v) for k, v in gs.items()}
        g1["event"] = g1["event"] - e
        h = g1["hits"].astype(np.int64)
        h0 = int(ev.zone_off[e * 24])
        g1["hits"] = np.where(h == 0xFFFFFFFF, h, h - h0).astype(np.uint32)
        r = compare_seeds(os_, g1)
        assert r["n_orc"] == r["n_gpu"] == r["n_common"] and r["bit_equal"], (e, r)
        n_s += r["n_common"]
        # long tracks of this event: (seed identity, velo, UT hits) sets
        ok = dict(zip(range(os_["n"]), seed_keys(os_["event"], os_["half"], os_["hits"], os_["state"])))
        gk = dict(zip((int(s) for s in g1["slot"]), seed_keys(g1["event"], g1["half"], g1["hits"], g1["state"])))
        lsel = gl["event"] == e
        l1 = {k: (v[lsel] if isinstance(v, np.ndarray) and v.shape[:1] == lsel.shape else v) for k, v in gl.items()}
        l1["velo"] = l1["velo"] - int(ev.velo_off[e])
        u = l1["ut"].astype(np.int64)
        l1["ut"] = np.where(u == 0xFFFFFFFF, u, u - int(ev.ut_off[e * 4])).astype(np.uint32)
        rl = compare_long(om, l1, ok, gk)
        assert rl["n_orc"] == rl["n_gpu"] == rl["n_common"] and rl["bit_equal"], (e, rl)
        n_l += rl["n_common"]
    assert n_s > 100 * len(sample) and n_l > 60 * len(sample)
    c.close()
