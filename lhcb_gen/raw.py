"""Raw (unsorted) view of generated events: the input of the event-preparation step.

Holds no reconstruction arithmetic: it only permutes the generator's hits inside each event with a seeded
shuffle and labels every hit with its zone (half * 12 + layer).
"""
import numpy as np


def shuffle_raw(ev, seed: int = 0):
    """Returns dict(raw_off u32[n_events+1], raw_x f32[n_hits], raw_zone u8[n_hits], src i64[n_hits]);
    src[k] = index in ev.hit_x of raw hit k."""
    rng = np.random.default_rng(seed)
    zo = ev.zone_off.astype(np.int64)
    n = int(zo[-1])
    zone_of_hit = np.repeat(np.arange(len(zo) - 1) % 24, np.diff(zo)).astype(np.uint8)
    raw_off = zo[::24].copy()
    src = np.empty(n, np.int64)
    for e in range(ev.n_events):
        b, t = raw_off[e], raw_off[e + 1]
        src[b:t] = b + rng.permutation(t - b)
    return dict(raw_off=raw_off.astype(np.uint32), raw_x=np.ascontiguousarray(ev.hit_x[src]),
                raw_zone=np.ascontiguousarray(zone_of_hit[src]), src=src)
