"""Parity of lhcb_prepare (event preparation, SURVEY 8(f)1 / PAPER.md L372) with oracle/prepare.py through
the C-ABI: index and byte work, so the bar is bit-exact equality of zone_off, hit_x and perm."""
import numpy as np
import pytest

from lhcb_gen import config, generate, shuffle_raw
from oracle.prepare import prepare as oracle_prepare

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx(geom):
    from paper_2606_14480_b200 import Context
    c = Context(geom)
    yield c
    c.close()


def gpu_prepare(ctx, raw_off, raw_x, raw_zone):
    t = ctx.torch
    up = lambda a, dt: t.from_numpy(np.ascontiguousarray(a, dt).view(np.int32 if dt == np.uint32 else dt)).to(ctx.dev)
    out = ctx.lhcb_prepare(up(raw_off, np.uint32), up(raw_x, np.float32), up(raw_zone, np.uint8))
    t.cuda.synchronize()
    return (out["zone_off"].cpu().numpy().view(np.uint32), out["hit_x"].cpu().numpy(),
            out["perm"].cpu().numpy().view(np.uint32), out["status"].cpu().numpy().view(np.uint32), out)


def check(ctx, raw_off, raw_x, raw_zone):
    zo, hx, pm, st, out = gpu_prepare(ctx, raw_off, raw_x, raw_zone)
    ozo, ohx, opm = oracle_prepare(raw_off, raw_x, raw_zone)
    assert not st.any()
    assert np.array_equal(zo, ozo)
    assert np.array_equal(hx.view(np.uint32), ohx.view(np.uint32))
    assert np.array_equal(pm, opm)
    return out


@pytest.mark.parametrize("cfg,n", [(1, 16), (2, 128), (4, 64)])
def test_prepare_equals_oracle(ctx, cfg, n):
    ev = generate(config(cfg, n))
    raw = shuffle_raw(ev, seed=cfg)
    check(ctx, raw["raw_off"], raw["raw_x"], raw["raw_zone"])
    assert ctx.last_launch_count() == 1


def test_prepare_edge_cases(ctx):
    rng = np.random.default_rng(11)
    # empty events, one-hit events, many equal x (ties -> stable by raw index), x outside the bin range,
    # -0.0 / +0.0, a single crowded zone
    sizes = np.array([0, 1, 0, 300, 2, 700, 0])
    raw_off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.uint32)
    n = int(raw_off[-1])
    x = np.round(rng.uniform(-4000, 4000, n), -1).astype(np.float32)
    x[5:40] = 0.0; x[40:60] = -0.0; x[60:80] = 12345.0; x[80:90] = -1e30
    zone = rng.integers(0, 24, n).astype(np.uint8)
    zone[int(raw_off[5]):int(raw_off[6])] = 17
    check(ctx, raw_off, x, zone)
    # zero events: no launch
    t = ctx.torch
    z = t.zeros(1, dtype=t.int32, device=ctx.dev)
    ctx.lhcb_prepare(z, t.zeros(0, device=ctx.dev), t.zeros(0, dtype=t.uint8, device=ctx.dev))
    assert ctx.last_launch_count() == 0


def test_prepare_crowded_cell(ctx):
    """More than 255 hits in one (zone, x-bin) cell (identical x, x within one bin, x outside the binned range):
    the kernel ranks such an event by all pairs; the order must still be the stable sort's."""
    rng = np.random.default_rng(12)
    sizes = np.array([900, 50, 1300, 0, 600])
    raw_off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.uint32)
    n = int(raw_off[-1])
    x = rng.uniform(-3000, 3000, n).astype(np.float32)
    zone = rng.integers(0, 24, n).astype(np.uint8)
    x[100:500] = 77.25; zone[100:500] = 5                      # 400 identical hits: ties by raw index
    b2 = int(raw_off[2])
    x[b2:b2 + 300] = rng.uniform(100.0, 101.0, 300).astype(np.float32); zone[b2:b2 + 300] = 9     # 300 hits inside one bin
    x[b2 + 300:b2 + 330] = 100.5
    b4 = int(raw_off[4])
    x[b4:b4 + 280] = rng.uniform(5000, 9000, 280).astype(np.float32); zone[b4:b4 + 280] = 23      # beyond the last bin
    check(ctx, raw_off, x, zone)


def test_prepare_other_instantiations_and_unaligned_outputs(ctx):
    """The largest event capacity (1,024 threads x 16 hits per thread) and output arrays that are not 16-byte
    aligned (scalar stores instead of the vector ones): same result as the oracle."""
    from lhcb_gen import default_geom
    from paper_2606_14480_b200 import Context
    ev = generate(config(4, 24))
    raw = shuffle_raw(ev, seed=21)
    c = Context(default_geom(max_hits_per_half=8000))
    check(c, raw["raw_off"], raw["raw_x"], raw["raw_zone"])
    c.close()
    t = ctx.torch
    up = lambda a, dt: t.from_numpy(np.ascontiguousarray(a, dt).view(np.int32 if dt == np.uint32 else dt)).to(ctx.dev)
    n_events, n = len(raw["raw_off"]) - 1, len(raw["raw_x"])
    hx = t.empty(n + 1, dtype=t.float32, device=ctx.dev)[1:]           # 4 bytes off a 16-byte boundary
    pm = t.empty(n + 3, dtype=t.int32, device=ctx.dev)[3:]
    out = dict(zone_off=t.empty(n_events * 24 + 1, dtype=t.int32, device=ctx.dev), hit_x=hx, perm=pm,
               status=t.empty(n_events, dtype=t.int32, device=ctx.dev))
    ctx.lhcb_prepare(up(raw["raw_off"], np.uint32), up(raw["raw_x"], np.float32), up(raw["raw_zone"], np.uint8), out)
    t.cuda.synchronize()
    ozo, ohx, opm = oracle_prepare(raw["raw_off"], raw["raw_x"], raw["raw_zone"])
    assert not out["status"].cpu().numpy().any()
    assert np.array_equal(out["zone_off"].cpu().numpy().view(np.uint32), ozo)
    assert np.array_equal(hx.cpu().numpy().view(np.uint32), ohx.view(np.uint32))
    assert np.array_equal(pm.cpu().numpy().view(np.uint32), opm)


def test_prepare_reports_bad_input_and_overflow(geom):
    from lhcb_gen import default_geom
    from paper_2606_14480_b200 import Context
    c = Context(default_geom(max_hits_per_half=512))
    ev = generate(config(2, 3))
    raw = shuffle_raw(ev, seed=1)
    x = raw["raw_x"].copy(); zone = raw["raw_zone"].copy()
    zo, hx, pm, st, _ = gpu_prepare(c, raw["raw_off"], x, zone)          # > 1024 raw hits per event
    assert (st == 8).all()
    # passed through unsorted, everything in zone 0 of its event
    assert np.array_equal(hx, x) and np.array_equal(pm, np.arange(len(x)))
    assert np.array_equal(zo[0::24], raw["raw_off"]) and np.array_equal(zo[1:24], np.full(23, raw["raw_off"][1]))
    c.close()
    c = Context(geom)
    x[int(raw["raw_off"][1]) + 5] = np.nan
    zone[int(raw["raw_off"][2]) + 7] = 24
    zo, hx, pm, st, _ = gpu_prepare(c, raw["raw_off"], x, zone)
    assert st.tolist() == [0, 512, 512]
    ozo, ohx, opm = oracle_prepare(raw["raw_off"][:2], x[:raw["raw_off"][1]], zone[:raw["raw_off"][1]])
    assert np.array_equal(zo[:25], ozo) and np.array_equal(pm[:len(opm)], opm)
    c.close()


def test_prepare_then_seeding_equals_seeding_on_sorted_input(ctx):
    """The prepared layout feeds lhcb_seeding: same seeds as from the generator's own sorted events."""
    from paper_2606_14480_b200 import DeviceEvents
    ev = generate(config(2, 32))
    raw = shuffle_raw(ev, seed=5)
    out = check(ctx, raw["raw_off"], raw["raw_x"], raw["raw_zone"])
    dev = DeviceEvents.from_host(ev)
    ref = ctx.seeds_to_host(ctx.lhcb_seeding(dev))
    dev.zone_off, dev.hit_x = out["zone_off"], out["hit_x"]
    got = ctx.seeds_to_host(ctx.lhcb_seeding(dev))
    assert ref["n"] == got["n"] > 100 * 32

    def canon(s):
        o = np.lexsort(tuple(s["hits"].T[::-1]) + (s["half"], s["event"]))
        return s["hits"][o], s["state"][o].view(np.uint32), s["par"][o].view(np.uint32)
    for a, b in zip(canon(ref), canon(got)):
        assert np.array_equal(a, b)


def test_prepare_full_size_cfg3(ctx):
    """BASELINE.json configs[2] at full size: properties that hold at any size + sampled events vs the oracle."""
    from paper_2606_14480_b200 import Context, capacities
    n = 16384
    ev = generate(config(3, n), workers=8)
    raw = shuffle_raw(ev, seed=9)
    c = Context(capacities.with_capacities(ev.geom))
    zo, hx, pm, st, _ = gpu_prepare(c, raw["raw_off"], raw["raw_x"], raw["raw_zone"])
    assert not st.any()
    assert np.array_equal(zo, ev.zone_off)                                   # the generator's layout comes back
    assert np.array_equal(hx.view(np.uint32), ev.hit_x.view(np.uint32))
    assert np.array_equal(raw["raw_x"][pm].view(np.uint32), hx.view(np.uint32))
    assert np.array_equal(np.sort(pm), np.arange(len(pm), dtype=np.uint32))  # a permutation
    ro = raw["raw_off"].astype(np.int64)
    for e in [0, 1, 4095, 8192, 16383] + list(range(7000, 7010)):
        ozo, ohx, opm = oracle_prepare(np.array([0, ro[e + 1] - ro[e]], np.uint32), raw["raw_x"][ro[e]:ro[e + 1]],
                                       raw["raw_zone"][ro[e]:ro[e + 1]])
        assert np.array_equal(pm[ro[e]:ro[e + 1]] - ro[e], opm)
    c.close()
