"""Pins of reading A15: every search window is CLOSED (a hit exactly on an edge is inside), the
cuts of Eq. 21 and chi2_match < 2 are strict, exact chi2 ties go to the lower index.

The events are built so that the edge values are exact in float64: a straight track at x = 0 (all fit parameters
exactly zero), so that a window centre is 0 and an edge is the window's half-width itself; the same IEEE
operations are done here and in the oracle.  A hit ON the edge must be taken, the next float64 beyond it must
not.  The observables are the oracle's own step counters and its candidate / seed lists."""
from types import SimpleNamespace

import numpy as np
import pytest

from lhcb_gen import default_geom
from oracle.binding import Oracle, NO_HIT

G = default_geom()


def event(hits_by_layer, half=0):
    """hits_by_layer: {layer: [x, ...]} of one event-half -> Events-like object (zones sorted)."""
    x, off = [], [0]
    for zone in range(24):
        h, l = divmod(zone, 12)
        xs = sorted(hits_by_layer.get(l, [])) if h == half else []
        x += xs
        off.append(len(x))
    x = np.array(x, np.float64)
    return SimpleNamespace(n_events=1, zone_off=np.array(off, np.uint32), hit_x=x.astype(np.float32), hit_x64=x,
                           polarity=np.array([-1], np.int8), geom=G)


def up(v):
    return float(np.nextafter(v, np.inf if v > 0 else -np.inf))      # the next float64 away from zero


def test_two_hit_and_three_hit_windows_are_closed():
    """Eq. 11 and the third-hit band (A4): T1 hit at x = 0, so the T3 window is [-dx3max, +dx3max] exactly; with the
    T3 hit at 0 as well the T2 band is [K d_hi, -K d_lo] exactly (K < 0)."""
    o = Oracle(G, "f64")
    c = o.constants()
    d3, K = float(c["dx3max"][0]), float(c["K"][0])
    d_lo, d_hi = G["cx_band"][2], G["cx_band"][3]
    assert K < 0
    # iteration 0: layers 0 (T1), 4 (T2), 8 (T3); iteration 1 has no hits
    s = o.seeding(event({0: [0.0], 8: [d3, -d3, up(d3), up(-d3)]}))
    assert s["counters"]["t1_hits"] == 1 and s["counters"]["pairs"] == 2
    hi2, lo2 = K * (-d_lo), K * d_hi                          # = x2c + K * cxlo, x2c + K * cxhi with x2c = 0, cx_pred = 0
    s = o.seeding(event({0: [0.0], 8: [0.0], 4: [hi2, lo2, up(hi2), up(lo2)]}))
    assert s["counters"]["pairs"] == 1 and s["counters"]["triplets"] == 2
    ev = event({0: [0.0], 8: [0.0], 4: [hi2, lo2, up(hi2), up(lo2)]})
    d = o.seeding_debug(ev, 0, 0)
    assert sorted(float(ev.hit_x64[i]) for i in d["t_idx"][:, 1]) == sorted([lo2, hi2])      # the two hits ON the edges


def test_extension_window_is_closed_and_the_cuts_are_as_written():
    """L90: +-1 mm around the prediction, closed.  Track at x = 0 (hits in layers 0, 4, 8, 7, 11), in layer 3 one
    hit exactly 1 mm away: attached; one float64 further: not.  (chi2 cut opened so that the candidate is listed.)"""
    g = default_geom(chi2x_max=1.0e12)
    o = Oracle(g, "f64")
    tol = g["tol_x_ext"]
    for x3, attached in ((tol, True), (-tol, True), (up(tol), False), (up(-tol), False)):
        ev = event({0: [0.0], 4: [0.0], 8: [0.0], 7: [0.0], 11: [0.0], 3: [x3]})
        d = o.seeding_debug(ev, 0, 0)
        it0 = d["c_it"] == 0
        assert it0.sum() == 1
        slot3 = 1                                             # x-layers in z order: 0, 3, 4, 7, 8, 11
        assert (d["c_hits"][it0][0][slot3] != NO_HIT) == attached, x3
        assert d["c_nx"][it0][0] == (6 if attached else 5)


def test_stereo_window_is_closed():
    """L215: +-2 mm around the stereo prediction, closed.  Track at x = 0, y = 0: every stereo prediction is 0.
    Five stereo hits at 0 and the sixth exactly 2 mm away is attached; one float64 further it is not."""
    g = default_geom(chi2y_max=1.0e12)
    o = Oracle(g, "f64")
    tol = g["tol_uv"]
    xl = {l: [0.0] for l in (0, 3, 4, 7, 8, 11)}
    for xs, n in ((tol, 6), (-tol, 6), (up(tol), 5), (up(-tol), 5)):
        hits = dict(xl); hits.update({l: [0.0] for l in (1, 2, 5, 6, 9)}); hits[10] = [xs]
        s = o.seeding(event(hits))
        assert s["n"] == 1 and s["nuv"][0] == n, (xs, s["nuv"])


def test_ut_loose_window_is_closed():
    """Table 2 loose window of the first UT layer, closed: VELO state on the z axis, q/p = 0, so the prediction is
    A_gamma dz^2 and the window half-width is the clamp value the oracle reports."""
    o = Oracle(G, "f64")
    w = o.ut_window(0, False, 0.0)
    dz = G["ut_z"][0] - G["z_velo"]
    centre = G["gamma_ab"][0] * (dz * dz)                     # (x_V + t_x dz) + gamma dz^2 - y tan(alpha), all else 0
    centre = (0.0 + 0.0 * dz) + centre
    x0e = centre - 0.0 * G["ut_tan_alpha"][0]
    off = np.array([0, 1, 1, 1, 1], np.uint32)
    for x, inside in ((x0e + w, True), (x0e - w, True), (up(x0e + w), False), (float(np.nextafter(x0e - w, -np.inf)), False)):
        r = o.ut_search([0.0, 0.0, 0.0, 0.0], 0.0, off, np.array([x]), np.array([-50.0]), np.array([50.0]))
        assert r["n"] == (1 if inside else 0), (x, r)


def test_equal_chi2_candidates_of_a_seed_go_to_the_lower_velo_index():
    """A14 / A15: one seed, two bit-identical VELO states: exactly equal chi2_match; the seed keeps the lower VELO
    index, and the pair is one long track, not two and not none."""
    o = Oracle(G, "f64")
    tx, ty = 0.03, -0.02
    velo = [2.0, -3.0, tx, ty]
    seed = [velo[0] + tx * (7826.0 - 770.0), velo[1] + ty * (7826.0 - 770.0), tx, ty, 0.0]
    ev = SimpleNamespace(n_events=1, polarity=np.array([-1], np.int8),
                         velo_off=np.array([0, 3], np.uint32), velo_x=np.array([50.0, velo[0], velo[0]]),
                         velo_y=np.array([40.0, velo[1], velo[1]]), velo_tx=np.array([0.2, tx, tx]), velo_ty=np.array([0.1, ty, ty]),
                         ut_off=np.zeros(5, np.uint32), ut_x0=np.zeros(0), ut_ylo=np.zeros(0), ut_yhi=np.zeros(0))
    m = o.matching(1, np.array([0, 1], np.uint32), np.array([seed]), ev, use_ut=False)
    assert m["n"] == 1 and int(m["seed"][0]) == 0 and int(m["velo"][0]) == 1


def test_first_layer_stereo_window_is_closed():
    """Eq. 16 / A19: track at x = 0, y = 0, so the first-layer window of stereo layer l is [-y_max tan, +y_half_tol tan]
    (upper half) exactly; hits ON both edges are first-layer hits (the oracle's uv_first counter), the next float64
    beyond them are not."""
    o = Oracle(G, "f64")
    xl = {l: [0.0] for l in (0, 3, 4, 7, 8, 11)}
    n_first = 0
    hits = dict(xl); hits.update({l: [0.0] for l in (1, 2, 5, 6, 9, 10)})
    for lf in G["uv_first_layer"]:
        ta = G["scifi_tan_alpha"][lf]
        a, b = 0.0 - (-G["y_half_tol"] * ta), 0.0 - (G["y_max"] * ta)       # x_pred - y tan(alpha) at both ends of the half
        hits[lf] = hits[lf] + [a, b, up(a), up(b)]
        n_first += 3                                                      # the track's own hit and the two edge hits
    s = o.seeding(event(hits))
    assert s["n"] == 1 and s["counters"]["xz_kept"] == 1
    assert s["counters"]["uv_first"] == n_first, s["counters"]["uv_first"]


def test_preselection_cuts_are_strict_on_every_variable(oracle64=None):
    """Eq. 21 as printed: |dx| < 20 mm, |dy| < 150 mm, |dtx| < 1.5 (|dty| < 0.02 is in test_oracle_constants).  With
    zero slopes dx = x_S - x_V and dy = y_S - y_V exactly; with t_x^V = 0, dtx = t_x^S exactly."""
    o = Oracle(G, "f64")
    below = lambda v: float(np.nextafter(v, 0.0))
    for seed, velo, ok in (([20.0, 0, 0, 0], [0, 0, 0, 0], 0.0), ([below(20.0), 0, 0, 0], [0, 0, 0, 0], 1.0),
                           ([0, 150.0, 0, 0], [0, 0, 0, 0], 0.0), ([0, below(150.0), 0, 0], [0, 0, 0, 0], 1.0),
                           ([-20.0, 0, 0, 0], [0, 0, 0, 0], 0.0), ([0, -150.0, 0, 0], [0, 0, 0, 0], 0.0)):
        r = o.match_pair([float(v) for v in seed], [float(v) for v in velo])
        assert r["presel"] == ok, (seed, r)
    # dtx: choose x_S so that dx = 0 at the z_match of this pair (fixed point on |x_S|), then dtx alone decides
    for dtx, ok in ((1.5, 0.0), (below(1.5), 1.0)):
        xs = 0.0
        for _ in range(40):
            zm = o.match_pair([xs, 0.0, dtx, 0.0], [0.0, 0.0, 0.0, 0.0])["zm"]
            xs = (7826.0 - zm) * dtx
        r = o.match_pair([xs, 0.0, dtx, 0.0], [0.0, 0.0, 0.0, 0.0])
        assert abs(r["dx"]) < 1.0 and r["dtx"] == dtx and r["presel"] == ok, (dtx, r)


def test_ut_strip_coverage_is_closed_at_the_tolerance():
    """Reading A18: a strip covers y if y_lo - 1 mm <= y <= y_hi + 1 mm, closed.  VELO state on the z axis (y = 0 at
    every layer): a strip starting exactly 1 mm above 0, or ending exactly 1 mm below, still covers it."""
    o = Oracle(G, "f64")
    tol = G["ut_y_tol"]
    dz = G["ut_z"][0] - G["z_velo"]
    x0e = (0.0 + 0.0 * dz) + G["gamma_ab"][0] * (dz * dz)
    off = np.array([0, 1, 1, 1, 1], np.uint32)
    for ylo, yhi, inside in ((tol, tol + 100.0, True), (up(tol), tol + 100.0, False), (-100.0 - tol, -tol, True),
                             (-100.0 - tol, up(-tol), False)):
        r = o.ut_search([0.0, 0.0, 0.0, 0.0], 0.0, off, np.array([x0e]), np.array([ylo]), np.array([yhi]))
        assert r["n"] == (1 if inside else 0), (ylo, yhi, r)


def test_hit_with_global_index_zero_is_a_hit_like_any_other():
    """Index 0 is a valid hit index (NO_HIT is 0xFFFFFFFF, "nothing found yet" is -1): (a) the first hit of the
    event is the closest one in its layer although a decoy 0.5 mm further sits at index 1; (b) with no hit in layer 0
    the first stereo hit has global index 0 and is attached like the others."""
    from tests.test_oracle_readings import make_event, track_hits, xz_track
    par = xz_track(p=13000.0, q=+1, tx0=0.01)
    hits = track_hits(par, lambda z: 0.02 * z)
    ev, idx = make_event(hits + [(0, 0, hits[0][2] + 0.5)])
    assert idx[0] == 0
    o = Oracle(G, "f64")
    d = o.seeding_debug(ev, 0, 0)
    it1 = d["c_it"] == 1                                      # iteration 1 reaches layer 0 by the +-1 mm extension
    assert it1.sum() == 1 and d["c_hits"][it1][0][0] == 0
    s = o.seeding(ev)
    assert s["n"] >= 1 and all(int(h[0]) == 0 for h in s["hits"])
    ev, idx = make_event([h for h in hits if h[1] != 0])
    assert idx[0] == 0 and ev.zone_off[1] == 0                # (position 0 of the list is now the layer-1 stereo hit)
    s = o.seeding(ev)
    assert s["n"] == 1 and s["nx"][0] == 5 and s["nuv"][0] == 6 and int(s["hits"][0][1]) == 0


def test_ut_strip_coverage_is_closed_in_the_tight_layers_too():
    o = Oracle(G, "f64")
    tol = G["ut_y_tol"]
    x0 = np.array([G["gamma_ab"][0] * ((z - G["z_velo"]) ** 2) for z in G["ut_z"]])      # q/p = 0: gamma_x = A_gamma
    off = np.array([0, 1, 2, 3, 4], np.uint32)
    for ylo2, n in ((tol, 4), (up(tol), 3)):
        ylo = np.array([-50.0, -50.0, ylo2, -50.0]); yhi = ylo + 100.0
        r = o.ut_search([0.0, 0.0, 0.0, 0.0], 0.0, off, x0, ylo, yhi)
        assert r["ok"] and r["n"] == n, (ylo2, r)
