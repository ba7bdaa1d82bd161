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


def test_cfg2_128_events(ctx, oracle32):
    ev = generate(config(2, 128))
    r, rl = check_chain(ctx, oracle32, ev, use_ut=True)
    assert r["n_common"] > 100 * 128 and rl["n_common"] > 60 * 128
    assert r["bit_equal"] and rl["bit_equal"]
    assert not r["only_orc"] and not r["only_gpu"] and not rl["only_orc"] and not rl["only_gpu"]


def test_cfg4_64_events(ctx, oracle32):
    ev = generate(config(4, 64))
    r, rl = check_chain(ctx, oracle32, ev, use_ut=True)
    assert r["bit_equal"] and rl["bit_equal"]
    assert not r["only_orc"] and not r["only_gpu"]


def test_cfg5_100_events(ctx, oracle32):
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


def test_twin_seeds_tie_is_decided_by_hit_lists(ctx, oracle32):
    """Reading A21 on the GPU: a twin of a matched seed (bit-identical state) is appended; whichever of the two
    hit lists comes first gets the long track, in either slot order, as in the oracle."""
    from paper_2606_14480_b200 import DeviceEvents
    ev = generate(config(5, 1))
    base = oracle32.matching(1, ev.seed_off, ev.seed_state.T, ev, use_ut=True)
    s0 = int(base["seed"][0]); n = ev.seed_state.shape[1]
    state = np.concatenate([ev.seed_state, ev.seed_state[:, s0:s0 + 1]], axis=1)
    off = np.array([0, n + 1], np.uint32)
    dev = DeviceEvents.from_host(ev)
    for twin_first in (False, True):
        hits = np.tile(np.arange(12, dtype=np.uint32), (n + 1, 1)) + 100 * np.arange(n + 1, dtype=np.uint32)[:, None]
        hits[n] = hits[s0]
        (hits[s0] if twin_first else hits[n])[7] += 1
        om = oracle32.matching(1, off, state.T, ev, use_ut=True, hits=hits)
        seeds, slot = ctx.seeds_from_states(1, off, state)
        t = ctx.torch
        h = np.full((12, seeds["cap_total"]), 0xFFFFFFFF, np.uint32)
        h[:, slot] = hits.T
        seeds["hits"] = t.from_numpy(h.view(np.int32)).to(ctx.dev)
        gl = ctx.long_to_host(ctx.lhcb_matching(seeds, dev, use_ut=True))
        inv = {int(sl): i for i, sl in enumerate(slot)}
        got = sorted((inv[int(a)], int(b)) for a, b in zip(gl["seed"], gl["velo"]))
        want = sorted((int(a), int(b)) for a, b in zip(om["seed"], om["velo"]))
        assert got == want
        assert ((n if twin_first else s0) in [g[0] for g in got]) and ((s0 if twin_first else n) not in [g[0] for g in got])
