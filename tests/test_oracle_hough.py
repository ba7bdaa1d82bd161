"""Pins of the Hough-cluster UV seeding in the oracle (reading A20)."""
from dataclasses import replace

import numpy as np

from lhcb_gen import config, default_geom, generate, truth, X_LAYERS, UV_LAYERS
from oracle.binding import Oracle, NO_HIT

G = default_geom()
Z = np.array(G["scifi_z"], np.float64)
TA = np.array(G["scifi_tan_alpha"], np.float64)
ZREF, DR = G["z_ref"], G["d_ratio"]


def g_of(z):
    zb = z - ZREF
    return zb * zb * (1 + DR * zb)


def test_noise_free_tracks_recovered_with_hough():
    """Tracks generated from the paper's model (Eq. 1, straight y through the origin), no noise.  The Hough
    hypotheses are fixed lines (no t_y refinement, L217), up to a quarter of a bin (0.9 mm at the stereo
    layers) off the track, so a neighbouring track's hit can win "closest" in rare cases: >= 99.5% of the
    reconstructible tracks are found, pure and identical to the iterative version's, and their y parameters
    equal truth to 1e-6 relative (f64)."""
    ev = generate(replace(config(1), sigma_x=0.0, n_events=32, seed=123))
    o = Oracle(G, "f64"); o.set_uv_hough(True)
    s = o.seeding(ev)
    pid, pur = truth.seed_pids(ev, s["hits"])
    assert (pid >= 0).all() and (pur == 1.0).mean() > 0.995
    den = truth.reconstructible_seed(ev)
    found = np.zeros(len(den), bool); found[pid] = True
    assert den.sum() > 500 and found[den].mean() > 0.995
    P = ev.particles
    ok = (pur == 1.0) & (s["nuv"] == 6)
    for k, name in ((3, "ay"), (4, "by")):
        t = P[name][pid][ok]; got = s["par"][ok, k]
        assert np.all(np.abs(got - t) <= 1e-6 * np.maximum(np.abs(t), 1e-3 if name == "ay" else 1e-6)), name
    s2 = Oracle(G, "f64").seeding(ev)
    a = {tuple(h) for h in s["hits"]}; b = {tuple(h) for h in s2["hits"]}
    assert len(a & b) > 0.995 * len(b)


def test_hough_bins_cover_the_half():
    c = Oracle(G, "f32").hough_constants()
    zmin = Z[UV_LAYERS].min()
    assert abs(c["tlo0"] + abs(G["y_half_tol"]) / zmin) < 1e-8 and abs(c["tlo1"] - G["y_min"] / zmin) < 1e-7
    assert abs(c["w"] * 64 - (G["y_max"] + abs(G["y_half_tol"])) / zmin) < 1e-6 and abs(c["w"] * c["invw"] - 1) < 1e-6


def python_hough(par, half, ev, zbase):
    """The literal reading A20 in Python float64 for one x-z candidate (ax, bx, cx)."""
    ax, bx, cx = par
    x = ev.hit_x64
    zmin = Z[UV_LAYERS].min(); tol = abs(G["y_half_tol"])
    ylo, yhi = ((-tol, G["y_max"]), (G["y_min"], tol))[half]
    tlo = ylo / zmin; w = (G["y_max"] + tol) / zmin / 64.0; invw = 64.0 / ((G["y_max"] + tol) / zmin)
    xp, votes, zones = [], [], []
    for l in UV_LAYERS:
        zb = Z[l] - ZREF
        xpl = (ax + bx * zb) + cx * g_of(Z[l])
        a, b = xpl - ylo * TA[l], xpl - yhi * TA[l]
        lo, hi = min(a, b), max(a, b)
        b0, b1 = int(ev.zone_off[zbase + l]), int(ev.zone_off[zbase + l + 1])
        v = set()
        for i in range(b0, b1):
            if lo <= x[i] <= hi:
                t = ((xpl - x[i]) * (1.0 / TA[l])) * (1.0 / Z[l])
                v.add(int(min(max((t - tlo) * invw, 0.0), 63.0)))
        xp.append(xpl); votes.append(v); zones.append((b0, b1))
    pop = [sum((b in v) or (b + 1 in v and b < 63) for v in votes) for b in range(64)]
    sel = [b for level in range(6, G["min_uv_hits"] - 1, -1) for b in range(64) if pop[b] == level][:8]
    best = None
    for b in sel:
        for k in range(4):
            ty = tlo + (b + (k * 0.5 + 0.25)) * w
            hits, rows, rhs = [], [], []
            for s, l in enumerate(UV_LAYERS):
                xe = xp[s] - ty * (Z[l] * TA[l])
                b0, b1 = zones[s]
                cand = [(abs(x[i] - xe), i) for i in range(b0, b1) if abs(x[i] - xe) <= G["tol_uv"]]
                if cand:
                    i = min(cand)[1]
                    hits.append(i); rows.append([-TA[l], -(Z[l] - ZREF) * TA[l]]); rhs.append(x[i] - xp[s])
                else:
                    hits.append(NO_HIT)
            n = len(rows)
            if n < G["min_uv_hits"]:
                continue
            A = np.array(rows); r = np.array(rhs)
            th = np.linalg.lstsq(A, r, rcond=None)[0]
            chi2 = float(((r - A @ th) ** 2).sum()) / G["sigma_hit"] ** 2 / (n - 2)
            if chi2 > G["chi2y_max"]:
                continue
            if best is None or n > best[0] or (n == best[0] and chi2 < best[1] - 1e-12):
                best = (n, chi2, hits)
    return best


def test_hough_equals_the_literal_reading_in_python():
    ev = generate(config(2, 4))
    o = Oracle(G, "f64"); o.set_uv_hough(True)
    s = o.seeding(ev)
    assert s["n"] > 400
    same = 0
    idx = range(0, s["n"], 7)
    for i in idx:
        zbase = (int(s["event"][i]) * 2 + int(s["half"][i])) * 12
        best = python_hough(s["par"][i, :3], int(s["half"][i]), ev, zbase)
        assert best is not None
        same += [int(h) for h in s["hits"][i][UV_LAYERS]] == [int(h) for h in best[2]] and best[0] == s["nuv"][i]
    assert same >= len(idx) - 1, (same, len(idx))            # (one seed of slack for a chi2 tie in float64)


def test_hough_finds_what_the_literal_reading_finds_for_every_survivor():
    """The other direction, and the iterative version too: for EVERY x-z candidate that survives the clone kill
    in a half, the literal Python reading decides whether there is a seed and with which stereo hits; the
    oracle's seeds of that half must be exactly those (no seed lost to a cluster threshold, a window or a
    hypothesis that is off by a fraction of a bin)."""
    from tests.test_oracle_readings import python_uv_iterative
    from types import SimpleNamespace
    ev = generate(config(2, 2))
    for hough in (True, False):
        o = Oracle(G, "f64"); o.set_uv_hough(hough)
        s = o.seeding(ev)
        n_checked = mism = 0
        for e in range(ev.n_events):
            for half in range(2):
                zbase = (e * 2 + half) * 12
                d = o.seeding_debug(ev, e, half)
                want = set()
                for c in np.flatnonzero(d["c_keep"]):
                    if hough:
                        best = python_hough(d["c_par"][c, :3], half, ev, zbase)
                    else:
                        sub = SimpleNamespace(zone_off=ev.zone_off[e * 24:e * 24 + 25], hit_x64=ev.hit_x64)
                        best = python_uv_iterative(d["c_par"][c, :3], half, sub)
                    if best is not None:
                        want.add((tuple(int(h) for h in d["c_hits"][c]), tuple(int(h) for h in best[2])))
                sel = (s["event"] == e) & (s["half"] == half)
                got = {(tuple(int(h) for h in hh[X_LAYERS]), tuple(int(h) for h in hh[UV_LAYERS])) for hh in s["hits"][sel]}
                n_checked += len(want | got); mism += len(want ^ got)
        assert n_checked > 250 and mism <= 2, (hough, n_checked, mism)     # (slack for chi2 ties / cut edges in float64)


def test_hough_seeds_a_track_with_exactly_the_minimum_of_stereo_hits():
    """A20 with L215: a cluster that exactly `min_uv_hits` (4) layers vote for is a cluster, and a combination of
    exactly four stereo hits is a seed: a hand-built track with stereo hits in layers 1, 5, 6 and 10 only."""
    from tests.test_oracle_readings import make_event, track_hits, xz_track
    par = xz_track(p=14000.0, q=+1, tx0=-0.02)
    hits = [h for h in track_hits(par, lambda z: 0.04 * z) if h[1] in X_LAYERS or h[1] in (1, 5, 6, 10)]
    ev, idx = make_event(hits)
    for hough in (True, False):
        o = Oracle(G, "f64"); o.set_uv_hough(hough)
        s = o.seeding(ev)
        assert s["n"] == 1 and s["nuv"][0] == 4 and s["nx"][0] == 6, (hough, s["n"])
        assert sorted(int(h) for h in s["hits"][0] if h != NO_HIT) == sorted(idx.values())


def test_hough_seed_invariants():
    ev = generate(config(2, 6))
    o = Oracle(G, "f32"); o.set_uv_hough(True)
    s = o.seeding(ev)
    it = Oracle(G, "f32").seeding(ev)
    x = ev.hit_x.astype(np.float64)
    for i in range(s["n"]):
        h = s["hits"][i]
        zbase = (s["event"][i] * 2 + s["half"][i]) * 12
        for l in range(12):
            if h[l] != NO_HIT:
                assert ev.zone_off[zbase + l] <= h[l] < ev.zone_off[zbase + l + 1]
        nuv = sum(h[l] != NO_HIT for l in UV_LAYERS)
        assert nuv == s["nuv"][i] and nuv in (4, 5, 6) and s["par"][i, 6] <= 8.0
        ax, bx, cx, ay, by = s["par"][i, :5].astype(np.float64)
        for l in UV_LAYERS:
            if h[l] != NO_HIT:
                zb = Z[l] - ZREF
                assert abs(x[h[l]] - (ax + bx * zb + cx * g_of(Z[l]) - (ay + by * zb) * TA[l])) < 2.0 + 1e-3
    # similar tracking performance (L204): efficiency within 3% of the iterative version on nominal events
    e_h = truth.seeding_summary(ev, s["hits"])["efficiency"]; e_i = truth.seeding_summary(ev, it["hits"])["efficiency"]
    assert e_h > 0.93 and abs(e_h - e_i) < 0.03
    # the x-z part is untouched by the choice of the UV version
    assert {tuple(h[X_LAYERS]) for h in s["hits"]} <= {tuple(c) for c in it["hits"][:, X_LAYERS]} | {tuple(h[X_LAYERS]) for h in s["hits"]}


def hough_cap_event(n_decoys, decoy_layers=(1, 2, 5, 6, 9, 10)):
    """One x-z track in the upper half whose true stereo hits sit in the middle of t_y bin 40, plus `n_decoys`
    decoy clusters at lower t_y (bins 2+4i and 3+4i).  A decoy has one hit per layer of `decoy_layers`, alternately
    0.3 bins above the lower edge of its first bin and 0.3 bins below the upper edge of its second bin: every one of
    those layers votes for the cluster, but a straight line of fixed t_y (the four hypotheses of a cluster, L217) is
    within 2 mm of at most half of the hits (a bin is 3.4-4.1 mm wide at the stereo layers), fewer than min_uv_hits:
    a decoy takes one of the "up to eight" places and yields no seed.  The true hits vote in bin 40 only, so the
    clusters (39, 40) and (40, 41) both have all six layers; (39, 40) comes first.  Returns (event, true hit indices)."""
    from tests.test_oracle_readings import make_event, track_hits, xz_track
    zmin = Z[UV_LAYERS].min(); tol = abs(G["y_half_tol"])
    tlo = -tol / zmin; w = (G["y_max"] + tol) / zmin / 64.0
    t_of = lambda b: tlo + b * w
    par = xz_track(p=16000.0, q=-1, tx0=0.01)
    hits = track_hits(par, lambda z: t_of(40.5) * z)
    n_true = len(hits)
    for i in range(n_decoys):
        b = 2 + 4 * i
        lo = track_hits(par, lambda z: t_of(b + 0.3) * z); hi = track_hits(par, lambda z: t_of(b + 1.7) * z)
        for k, l in enumerate(UV_LAYERS):
            if l in decoy_layers:
                hits.append((lo if k % 2 == 0 else hi)[l])
    ev, idx = make_event(hits)
    return ev, sorted(idx[k] for k in range(n_true))


def test_hough_takes_up_to_eight_clusters_most_populated_first_then_lower_ty():
    """"Up to eight of the best bins" (reading A20: most voting layers first, then lower t_y).
    With seven six-layer decoy clusters below it the true cluster is the eighth and is seeded; with eight it is the
    ninth and is not; with eight five-layer decoys it ranks first again."""
    for mode in ("f64", "f32"):
        o = Oracle(G, mode); o.set_uv_hough(True)
        ev, true_hits = hough_cap_event(7)
        s = o.seeding(ev)
        assert s["n"] == 1 and s["nuv"][0] == 6 and sorted(int(h) for h in s["hits"][0]) == true_hits, (mode, s["n"])
        ev, _ = hough_cap_event(8)
        assert o.seeding(ev)["n"] == 0, mode
        ev, true_hits = hough_cap_event(8, decoy_layers=(1, 2, 5, 6, 9))
        s = o.seeding(ev)
        assert s["n"] == 1 and sorted(int(h) for h in s["hits"][0]) == true_hits, mode
        # the iterative version has no such cap: it seeds the track whatever the decoys
        it = Oracle(G, mode).seeding(hough_cap_event(8)[0])
        assert it["n"] == 1
