"""ORACLE (test infrastructure only; never imported by the product path) of the event preparation that
precedes the Seeding: raw, unsorted SciFi hits -> the tiled, sorted layout the paper assumes.

PAPER.md L372 (section 5.2): hits are "tiled by detector half" (y > 0 / y < 0), split per layer, and the
searches of section 3 need them sorted in x inside each (half, layer) zone.
makes this the step before the hot path.  The definition is a plain stable sort:

    inside every event, order the hits by (zone, x, raw index),   zone = half * 12 + layer

`zone_off` is the prefix sum of the per-zone counts, `hit_x` the x in that order and `perm[k]` the raw index
of sorted hit k.  numpy.lexsort is the library primitive; there is no blocking or reordering.  Pins
(tests/test_oracle_prepare.py): a hand-worked example (tests/golden/prepare_example.txt), a pure-Python
insertion sort on small inputs, permutation / sortedness / stability invariants, and the round trip
"shuffle the generator's events, prepare them, get the generator's layout back".
"""
import numpy as np

N_ZONES = 24


def prepare(raw_off, raw_x, raw_zone):
    """raw_off u32[n_events+1]; raw_x f32[n_hits]; raw_zone u8[n_hits] in [0, 24).
    Returns (zone_off u32[n_events*24+1], hit_x f32[n_hits], perm u32[n_hits])."""
    raw_off = np.asarray(raw_off, np.int64)
    raw_x = np.asarray(raw_x, np.float32)
    raw_zone = np.asarray(raw_zone, np.int64)
    n_events = len(raw_off) - 1
    zone_off = np.zeros(n_events * N_ZONES + 1, np.int64)
    hit_x = np.empty_like(raw_x)
    perm = np.empty(len(raw_x), np.int64)
    for e in range(n_events):
        b, t = raw_off[e], raw_off[e + 1]
        x, z = raw_x[b:t], raw_zone[b:t]
        order = np.lexsort((np.arange(t - b), x, z))        # last key is the primary one
        hit_x[b:t] = x[order]
        perm[b:t] = b + order
        counts = np.bincount(z, minlength=N_ZONES)
        zone_off[e * N_ZONES + 1:(e + 1) * N_ZONES + 1] = b + np.cumsum(counts)
    zone_off[0] = raw_off[0]
    return zone_off.astype(np.uint32), hit_x, perm.astype(np.uint32)
