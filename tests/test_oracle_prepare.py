"""Pins of the event-preparation oracle (oracle/prepare.py): PAPER.md L372, SURVEY.md 8(f)1."""
import os

import numpy as np

from lhcb_gen import config, generate, shuffle_raw
from oracle.prepare import prepare

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "prepare_example.txt")


def read_golden():
    raw, out = [], {}
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#") or line == "raw":
            continue
        f = line.split()
        if f[0] in ("perm", "hit_x", "zone_off"):
            out[f[0]] = f[1:]
        else:
            raw.append((int(f[0]), int(f[1]), float(f[2])))
    return raw, out


def test_hand_worked_example():
    raw, exp = read_golden()
    ev = np.array([r[0] for r in raw]); zone = np.array([r[1] for r in raw], np.uint8)
    x = np.array([r[2] for r in raw], np.float32)
    raw_off = np.concatenate([[0], np.cumsum(np.bincount(ev))]).astype(np.uint32)
    zone_off, hit_x, perm = prepare(raw_off, x, zone)
    assert perm.tolist() == [int(v) for v in exp["perm"]]
    assert hit_x.tolist() == [float(v) for v in exp["hit_x"]]
    for item in exp["zone_off"]:
        k, v = item.split("=")
        if k == "end":
            assert zone_off[-1] == int(v)
        else:
            e, z = map(int, k.split(":"))
            assert zone_off[e * 24 + z] == int(v), item


def insertion_sort_reference(raw_off, x, zone):
    """Literal definition, pure Python: insertion sort (stable) on the key (zone, x) per event."""
    perm = []
    for e in range(len(raw_off) - 1):
        order = []
        for i in range(int(raw_off[e]), int(raw_off[e + 1])):
            k = len(order)
            while k > 0 and (zone[order[k - 1]], x[order[k - 1]]) > (zone[i], x[i]):
                k -= 1
            order.insert(k, i)
        perm += order
    return perm


def test_equals_insertion_sort_on_small_random_inputs():
    rng = np.random.default_rng(7)
    for trial in range(20):
        n_ev = int(rng.integers(1, 5))
        sizes = rng.integers(0, 60, n_ev)
        raw_off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.uint32)
        n = int(raw_off[-1])
        x = np.round(rng.uniform(-50, 50, n), 0).astype(np.float32)      # many ties
        zone = rng.integers(0, 24 if trial % 2 else 3, n).astype(np.uint8)
        zone_off, hit_x, perm = prepare(raw_off, x, zone)
        assert perm.tolist() == insertion_sort_reference(raw_off, x, zone)
        assert np.array_equal(hit_x, x[perm])
        cnt = np.diff(zone_off.astype(np.int64))
        for e in range(n_ev):
            assert np.array_equal(cnt[e * 24:(e + 1) * 24], np.bincount(zone[raw_off[e]:raw_off[e + 1]], minlength=24))


def test_invariants_and_round_trip_with_the_generator():
    ev = generate(config(2, 6))
    raw = shuffle_raw(ev, seed=3)
    zone_off, hit_x, perm = prepare(raw["raw_off"], raw["raw_x"], raw["raw_zone"])
    # the generator's layout comes back exactly
    assert np.array_equal(zone_off, ev.zone_off)
    assert np.array_equal(hit_x.view(np.uint32), ev.hit_x.view(np.uint32))
    # perm is a permutation inside each event and maps back to the generator's hits (up to equal x)
    assert np.array_equal(np.sort(perm), np.arange(len(perm)))
    assert np.array_equal(ev.hit_x[raw["src"][perm]], ev.hit_x)
    zo = zone_off.astype(np.int64)
    for z in range(len(zo) - 1):
        seg = hit_x[zo[z]:zo[z + 1]]
        assert (np.diff(seg) >= 0).all()
        ties = np.flatnonzero(np.diff(seg) == 0)
        assert (perm[zo[z] + ties] < perm[zo[z] + ties + 1]).all()       # stable
    # empty events and an empty batch
    z0, h0, p0 = prepare(np.zeros(3, np.uint32), np.zeros(0, np.float32), np.zeros(0, np.uint8))
    assert len(z0) == 49 and not z0.any() and len(h0) == 0 and len(p0) == 0
