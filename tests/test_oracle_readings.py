"""Pins of four oracle behaviours that the closed forms, brute force and invariants do not see
("What's weak" 1): each test fails when the one line of oracle/oracle.c that implements the
behaviour is changed.

  * O8 / reading A7  (the t_y estimate is "refined by averaging" with every new stereo hit)
  * O13              (in the tight windows "the closest hit ... is attached")
  * reading A19      (the halves overlap slightly: first-layer window y in [-y_half_tol, y_max])
  * reading A15      (closest-hit ties go to the lower hit index), for the +-1 mm x extension (L90), the
                     +-2 mm stereo search (L215) and the UT tight window (L309)
  * reading A21      (exact chi2_match ties between twin seeds are broken by their hit lists, not their order)

The events are built by hand from the paper's track model (Eq. 1, straight line in y), so what must come out
is known from the geometry; the t_y rule is also re-derived literally in Python float64.
"""
from types import SimpleNamespace

import numpy as np
import pytest

from lhcb_gen import default_geom, X_LAYERS, UV_LAYERS
from oracle.binding import Oracle, NO_HIT

G = default_geom()
Z = np.array(G["scifi_z"], np.float64)
TA = np.array(G["scifi_tan_alpha"], np.float64)
ZREF, DR = G["z_ref"], G["d_ratio"]
POL = -1


def g_of(z):
    zb = z - ZREF
    return zb * zb * (1 + DR * zb)


def xz_track(p=10000.0, q=+1, tx0=0.05):
    """(ax, bx, cx) of a prompt track of the toy model: kick K_B/p at z_match, Eq. 1 inside the SciFi."""
    A, B, C, D, E = G["mag"]
    dtx = POL * q * G["kick_pt"] / p
    tx_s = tx0 + dtx
    x_s = tx0 * G["z_scifi_state"]
    for _ in range(20):
        zm = A + B * abs(dtx) + C * dtx * dtx + D * abs(x_s) + E * tx0 * tx0
        x_s = zm * tx0 + (G["z_scifi_state"] - zm) * tx_s
    cx = POL * q * G["kappa_cx"] / p
    zbs = G["z_scifi_state"] - ZREF
    bx = tx_s - cx * (2 * zbs + 3 * DR * zbs * zbs)
    ax = x_s - bx * zbs - cx * g_of(G["z_scifi_state"])
    return ax, bx, cx


def track_hits(par, y_of_z, half=0):
    """One hit per layer from Eq. 1 and y(z): list of (half, layer, x)."""
    ax, bx, cx = par
    return [(half, l, ax + bx * (Z[l] - ZREF) + cx * g_of(Z[l]) - y_of_z(Z[l]) * TA[l]) for l in range(12)]


def make_event(hits):
    """hits: list of (half, layer, x) of ONE event -> Events-like object (sorted zones) + index lookup."""
    hits = sorted(enumerate(hits), key=lambda t: (t[1][0] * 12 + t[1][1], t[1][2], t[0]))
    x = np.array([h[2] for _, h in hits], np.float64)
    zone = np.array([h[0] * 12 + h[1] for _, h in hits], np.int64)
    off = np.zeros(25, np.uint32)
    np.cumsum(np.bincount(zone, minlength=24), out=off[1:])
    index_of = {orig: pos for pos, (orig, _) in enumerate(hits)}       # input position -> global hit index
    ev = SimpleNamespace(n_events=1, zone_off=off, hit_x=x.astype(np.float32), hit_x64=x,
                         polarity=np.array([POL], np.int8), geom=G)
    return ev, index_of


# --------------------------------------------------------------------------------------- O8 / A7
def python_uv_iterative(par, half, ev, update=True):
    """O8 + O9 written out literally in Python float64 for one x-z candidate (Eq. 16):
    returns (n, chi2y, stereo hit indices in UV_LAYERS order) of the best combination or None."""
    ax, bx, cx = par
    x = ev.hit_x64
    tol = G["y_half_tol"]
    ylo, yhi = ((-tol, G["y_max"]), (G["y_min"], tol))[half]
    xp = {l: (ax + bx * (Z[l] - ZREF)) + cx * g_of(Z[l]) for l in UV_LAYERS}
    zone = {l: (int(ev.zone_off[half * 12 + l]), int(ev.zone_off[half * 12 + l + 1])) for l in UV_LAYERS}
    best = None
    for lf in G["uv_first_layer"]:
        a, b = xp[lf] - ylo * TA[lf], xp[lf] - yhi * TA[lf]
        for ih in range(*zone[lf]):
            if not (min(a, b) <= x[ih] <= max(a, b)):
                continue
            ty = ((xp[lf] - x[ih]) / TA[lf]) / Z[lf]                       # Eq. 16, t_y = y / z
            got = {lf: ih}
            for l in UV_LAYERS:
                if l == lf:
                    continue
                xe = xp[l] - ty * Z[l] * TA[l]
                cand = [(abs(x[i] - xe), i) for i in range(*zone[l]) if abs(x[i] - xe) <= G["tol_uv"]]
                if cand:
                    i = min(cand)[1]
                    got[l] = i
                    if update:
                        ty = 0.5 * (ty + ((xp[l] - x[i]) / TA[l]) / Z[l])   # L215: refined by averaging
            n = len(got)
            if n < G["min_uv_hits"]:
                continue
            A = np.array([[-TA[l], -(Z[l] - ZREF) * TA[l]] for l in got])
            r = np.array([x[i] - xp[l] for l, i in got.items()])
            th = np.linalg.lstsq(A, r, rcond=None)[0]
            chi2 = float(((r - A @ th) ** 2).sum()) / G["sigma_hit"] ** 2 / (n - 2)
            if chi2 > G["chi2y_max"]:
                continue
            if best is None or n > best[0] or (n == best[0] and chi2 < best[1] - 1e-12):
                best = (n, chi2, [got.get(l, NO_HIT) for l in UV_LAYERS])
    return best


def test_ty_running_average_decides_the_stereo_hits():
    """Tracks whose straight line in y does not point to the origin (a displaced vertex: y = c + t z):
    t_y = y/z changes from layer to layer, and only the running average of L215 keeps the prediction within
    the 2 mm window.  The oracle's seeds equal the literal Python walk; without the averaging step that
    walk gives different hits for part of the tracks (so the test sees a dropped update)."""
    o = Oracle(G, "f64")
    differs = 0
    cases = [(c, t) for c in (0.0, 120.0, 200.0, 240.0, 270.0, 300.0, 330.0) for t in (0.02, 0.07)]
    for k, (c, t) in enumerate(cases):
        par = xz_track(p=8000.0 + 1500.0 * k, q=(-1) ** k, tx0=0.03 * (k % 5 - 2))
        hits = track_hits(par, lambda z: c + t * z)
        # decoys 1.5 mm beside the true stereo hits: "closest" must still pick the true ones
        hits += [(0, l, x + 1.5) for (_, l, x) in hits if l in (5, 9)]
        ev, _ = make_event(hits)
        s = o.seeding(ev)
        want = python_uv_iterative(par, 0, ev, update=True)
        no_upd = python_uv_iterative(par, 0, ev, update=False)
        differs += (want is None) != (no_upd is None) or (want is not None and want[2] != no_upd[2])
        if want is None:
            assert s["n"] == 0, (c, t)
            continue
        assert s["n"] == 1, (c, t, s["n"])
        assert [int(h) for h in s["hits"][0][UV_LAYERS]] == want[2] and s["nuv"][0] == want[0], (c, t)
        assert s["par"][0, 6] == pytest.approx(want[1], rel=1e-6, abs=1e-9)
    assert differs >= 3, "the cases no longer separate the averaged t_y from a fixed one"


def test_uv_walk_equals_the_literal_reading_on_displaced_events():
    """The same literal walk on generated high-occupancy events with displaced tracks (BASELINE.json
    configs[3]): every 5th seed of the f64 oracle, from its own x-z parameters."""
    from lhcb_gen import config, generate
    ev = generate(config(4, 3))
    s = Oracle(G, "f64").seeding(ev)
    assert s["n"] > 300
    idx = range(0, s["n"], 5)
    same = 0
    for i in idx:
        e, h = int(s["event"][i]), int(s["half"][i])
        z0 = e * 24
        sub = SimpleNamespace(zone_off=ev.zone_off[z0:z0 + 25], hit_x64=ev.hit_x64)
        best = python_uv_iterative(s["par"][i, :3], h, sub)
        same += best is not None and [int(x) for x in s["hits"][i][UV_LAYERS]] == best[2] and best[0] == s["nuv"][i]
    assert same >= 0.99 * len(idx), (same, len(idx))       # 1%: chi2 ties / cut edges in float64


# --------------------------------------------------------------------------------------- A19
def test_half_overlap_keeps_a_track_at_the_edge_of_its_half():
    """A track of the upper half at y = +1 mm whose two first-layer stereo hits are measured 0.26 mm off,
    i.e. at y0 = -2 mm: outside y >= 0, inside the overlap of reading A19 ([-5 mm, y_max]).  Only the
    overlap lets the stereo search start; the seed then carries all twelve hits."""
    par = xz_track(p=12000.0, tx0=-0.04)
    hits = track_hits(par, lambda z: 1.0)
    for l in G["uv_first_layer"]:
        h, ll, x = hits[l]
        hits[l] = (h, ll, x + 3.0 * TA[l])                   # y0 = (x_pred - x) / tan(alpha) = 1 - 3 = -2 mm
    ev, idx = make_event(hits)
    for mode in ("f64", "f32"):
        s = Oracle(G, mode).seeding(ev)
        assert s["n"] == 1 and s["nx"][0] == 6 and s["nuv"][0] == 6, mode
        assert [int(v) for v in s["hits"][0]] == [idx[l] for l in range(12)]
    # and the window does end at -y_half_tol: at y0 = -7 mm the track is not seeded from that layer
    hits = track_hits(par, lambda z: 1.0)
    for l in G["uv_first_layer"]:
        h, ll, x = hits[l]
        hits[l] = (h, ll, x + 8.0 * TA[l])
    ev, _ = make_event(hits)
    assert Oracle(G, "f64").seeding(ev)["n"] == 0


def test_first_layer_window_spans_the_half_plus_the_overlap():
    """Eq. 16 / reading A19 in numbers: the first-layer stereo window of an x-z candidate holds exactly the hits
    with y = (x_pred - x) / tan(alpha) in [-y_half_tol, y_max] (upper half; mirrored [y_min, +y_half_tol] in the
    lower one).  Decoys 1 mm inside and 1 mm outside of each edge, in both first layers: the oracle's own step
    counter of first-layer hits (uv_first) must count the track's hit and the two inner decoys per pass."""
    par = xz_track(p=15000.0, tx0=0.02)
    ax, bx, cx = par
    tol, ymax, ymin = G["y_half_tol"], G["y_max"], G["y_min"]
    for half, sign, edges in ((0, +1.0, (-tol, ymax)), (1, -1.0, (ymin, tol))):
        hits = track_hits(par, lambda z: sign * 40.0, half=half)
        inside = outside = 0
        for lf in G["uv_first_layer"]:
            xp = ax + bx * (Z[lf] - ZREF) + cx * g_of(Z[lf])
            for edge, inward in ((edges[0], +1.0), (edges[1], -1.0)):
                hits.append((half, lf, xp - (edge + inward * 1.0) * TA[lf])); inside += 1
                hits.append((half, lf, xp - (edge - inward * 1.0) * TA[lf])); outside += 1
        ev, _ = make_event(hits)
        s = Oracle(G, "f64").seeding(ev)
        assert s["n"] == 1 and s["nuv"][0] == 6, half
        assert s["counters"]["xz_kept"] == 1
        assert s["counters"]["uv_first"] == 2 + inside, (half, s["counters"]["uv_first"])     # 2 = the track's own hits


def test_more_stereo_hits_beat_an_earlier_combination():
    """L215 / L219: among the combinations of one x-z candidate the one with more stereo hits wins, whatever the
    order they are found in.  Two straight lines in y share the x-z track: line A (t_y = 0.05) has four stereo hits
    (layers 1, 2, 5, 6), line B (t_y = 0.03) all six.  In the first pass A's hit comes first (lower x in the u
    layer), so B has to replace it; the seed carries B's six hits."""
    par = xz_track(p=11000.0, q=-1, tx0=0.03)
    hits_b = track_hits(par, lambda z: 0.03 * z)
    hits_a = [h for h in track_hits(par, lambda z: 0.05 * z) if h[1] in (1, 2, 5, 6)]
    assert hits_a[0][2] < hits_b[1][2]                       # A's first-layer hit is met first
    ev, idx = make_event(hits_b + hits_a)
    for mode in ("f64", "f32"):
        s = Oracle(G, mode).seeding(ev)
        assert s["n"] == 1 and s["nuv"][0] == 6, (mode, s["n"], s["nuv"])
        assert [int(v) for v in s["hits"][0]] == [idx[l] for l in range(12)]
    # ... and with equal numbers of hits the better chi2 wins: B's hits smeared, A complete and exact
    rng = np.random.default_rng(5)
    hits_b2 = [(h, l, x + (0.25 * rng.standard_normal() if l in UV_LAYERS else 0.0)) for (h, l, x) in hits_b]
    hits_a2 = [h for h in track_hits(par, lambda z: 0.05 * z) if h[1] in UV_LAYERS]
    ev, idx = make_event(hits_b2 + hits_a2)
    s = Oracle(G, "f64").seeding(ev)
    assert s["n"] == 1 and s["nuv"][0] == 6
    assert [int(s["hits"][0][l]) for l in UV_LAYERS] == [idx[12 + k] for k in range(6)]      # line A's hits


# --------------------------------------------------------------------------------------- A15
def test_closest_hit_ties_go_to_the_lower_index():
    """Two hits at exactly the same x inside the +-1 mm window of the x extension (layer 3, searched by
    iteration 0) and inside the +-2 mm stereo window (layer 5): the lower index is attached."""
    par = xz_track(p=9000.0, q=-1, tx0=0.06)
    hits = track_hits(par, lambda z: 0.03 * z)
    hits += [hits[3], hits[5]]                               # exact duplicates (same float64 and float32 x)
    ev, idx = make_event(hits)
    lo3, lo5 = idx[3], idx[5]                                # make_event keeps input order among equal x
    assert idx[12] == lo3 + 1 and idx[13] == lo5 + 1
    for mode in ("f64", "f32"):
        o = Oracle(G, mode)
        d = o.seeding_debug(ev, 0, 0)
        it0 = d["c_it"] == 0
        assert it0.sum() == 1 and d["c_hits"][it0][0][X_LAYERS.index(3)] == lo3      # extension: lower index
        s = o.seeding(ev)
        assert s["n"] >= 1
        assert all(int(h[5]) == lo5 for h in s["hits"])                              # stereo: lower index


def test_ut_tight_window_takes_the_closest_hit_and_ties_go_low():
    """O13: a decoy 0.3 mm below the true hit sits at the lower index inside the tight window (0.5 mm at
    5 GeV, Table 2); the closest hit (the true one) is attached.  Two hits at the same x0: lower index."""
    from tests.test_oracle_matching import make_ut, AG, BG
    o = Oracle(G, "f64")
    qop = 1 / 5000.0
    gamma = AG + BG * qop
    velo = [3.0, -4.0, 0.04, -0.03]
    off, x0, ylo, yhi, tidx = make_ut(velo, gamma, extra=[(1, -0.3), (2, -0.3), (3, -0.3)])
    for l in (1, 2, 3):
        assert x0[tidx[l] - 1] == pytest.approx(x0[tidx[l]] - 0.3)     # the decoy precedes the true hit
    r = o.ut_search(velo, qop, off, x0, ylo, yhi)
    assert r["ok"] and r["n"] == 4 and (r["idx"] == tidx).all()
    assert r["gamma"] == pytest.approx(gamma, rel=1e-9)
    # exact duplicate of the true hit in a tight-window layer: the lower of the two indices
    off, x0, ylo, yhi, tidx = make_ut(velo, gamma, extra=[(2, 0.0)])
    assert x0[tidx[2]] == x0[tidx[2] - 1] or x0[tidx[2]] == x0[tidx[2] + 1]
    lo = tidx[2] - 1 if x0[tidx[2]] == x0[tidx[2] - 1] else tidx[2]
    r = o.ut_search(velo, qop, off, x0, ylo, yhi)
    assert r["ok"] and r["idx"][2] == lo


# --------------------------------------------------------------------------------------- A21
def test_twin_seeds_tie_is_broken_by_hit_lists_not_by_order():
    """Two seeds with bit-identical states (twins from a duplicate hit) and one VELO partner: whatever the
    order of the two seeds, the long track goes to the seed whose hit list comes first (reading A21)."""
    from lhcb_gen import config, generate
    ev = generate(config(5, 1))
    o = Oracle(G, "f32")
    base = o.matching(1, ev.seed_off, ev.seed_state.T, ev, use_ut=True)
    assert base["n"] > 50
    s0 = int(base["seed"][0])
    n = ev.seed_state.shape[1]
    state = np.concatenate([ev.seed_state.T, ev.seed_state.T[s0:s0 + 1]])          # twin of s0 appended
    off = np.array([0, n + 1], np.uint32)
    hits = np.tile(np.arange(12, dtype=np.uint32), (n + 1, 1)) + 100 * np.arange(n + 1, dtype=np.uint32)[:, None]
    for twin_first in (False, True):
        h = hits.copy()
        h[s0], h[n] = h[s0].copy(), h[s0].copy()
        (h[s0] if twin_first else h[n])[7] += 1                                     # the later twin: duplicate hit, index + 1
        want = n if twin_first else s0
        m = o.matching(1, off, state, ev, use_ut=True, hits=h)
        used = set(int(x) for x in m["seed"])
        assert want in used and (s0 + n - want) not in used
        assert m["n"] == base["n"]
    # without hit lists the lower seed index wins (direct seeds, BASELINE.json configs[4])
    m = o.matching(1, off, state, ev, use_ut=True)
    assert s0 in set(int(x) for x in m["seed"]) and n not in set(int(x) for x in m["seed"])
