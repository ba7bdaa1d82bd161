"""Pins of the oracle's matching steps O11..O14 (closed forms are in test_oracle_constants.py)."""
import numpy as np
import pytest

from lhcb_gen import config, default_geom, generate, truth
from oracle.binding import Oracle, NO_HIT

UT_Z = np.array([2327.0, 2372.0, 2597.0, 2642.0])
UT_TAN = np.array(default_geom()["ut_tan_alpha"])
AG, BG = 7.707063e-11, -7.817364e-3


def make_ut(velo, gamma, extra=()):
    """UT hits generated exactly from PAPER.md Eq. 19 (no pitch quantisation), one per layer, plus
    optional decoys (layer, dx0).  Returns ut_off[5], x0, ylo, yhi sorted per layer and the true indices."""
    x, y, tx, ty = velo
    lay, x0, ylo, yhi, is_true = [], [], [], [], []
    for i in range(4):
        dz = UT_Z[i] - 770.0
        yy = y + ty * dz
        xx = x + tx * dz + gamma * dz * dz
        lay.append(i); x0.append(xx - yy * UT_TAN[i]); ylo.append(np.floor(yy / 100) * 100)
        yhi.append(ylo[-1] + 100); is_true.append(True)
        for (li, d) in extra:
            if li == i:
                lay.append(i); x0.append(x0[-1 if not is_true[-1] else -1] + d)
                ylo.append(ylo[-1]); yhi.append(yhi[-1]); is_true.append(False)
    lay, x0, ylo, yhi, is_true = map(np.array, (lay, x0, ylo, yhi, is_true))
    order = np.lexsort((x0, lay))
    off = np.zeros(5, np.uint32); np.cumsum(np.bincount(lay, minlength=4), out=off[1:])
    true_idx = np.full(4, NO_HIT, np.uint32)
    for pos, j in enumerate(order):
        if is_true[j]:
            true_idx[lay[j]] = pos
    return off, x0[order], ylo[order], yhi[order], true_idx


def test_ut_noise_free_recovery(oracle64):
    """All four noise-free UT hits attached and gamma (hence q/p, Eq. 20) recovered to 1e-6 even when
    the kick estimate of q/p is 3% off (SURVEY 8(c) pin of O13)."""
    rng = np.random.default_rng(1)
    for _ in range(50):
        qop = rng.choice([-1, 1]) / np.exp(rng.uniform(np.log(3000), np.log(50000)))
        gamma = AG + BG * qop
        velo = [rng.uniform(-20, 20), rng.uniform(-20, 20), rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2)]
        off, x0, ylo, yhi, tidx = make_ut(velo, gamma, extra=[(1, 3.5), (2, -6.0), (3, 5.0)])
        r = oracle64.ut_search(velo, qop * 1.03, off, x0, ylo, yhi)
        assert r["ok"] and r["n"] == 4 and (r["idx"] == tidx).all()
        assert r["gamma"] == pytest.approx(gamma, rel=1e-9)
        assert (r["gamma"] - AG) / BG == pytest.approx(qop, rel=1e-6)
        assert r["ssq"] < 1e-16


def test_ut_loose_then_tight_and_min_hits(oracle64):
    qop = 1 / 5000.0
    gamma = AG + BG * qop
    velo = [1.0, -2.0, 0.05, 0.02]
    off, x0, ylo, yhi, tidx = make_ut(velo, gamma)
    # drop the first-layer hit: the loose search moves on to UTaU and still finds three hits (L311)
    keep = np.ones(4, bool); keep[tidx[0]] = False
    off2 = off.copy(); off2[1:] -= 1
    r = oracle64.ut_search(velo, qop, off2, x0[keep], ylo[keep], yhi[keep])
    assert r["ok"] and r["n"] == 3 and r["idx"][0] == NO_HIT
    # drop two: fewer than three hits -> rejected ("more than two", L311)
    keep[tidx[2]] = False
    off3 = off2.copy(); off3[3:] -= 1
    r = oracle64.ut_search(velo, qop, off3, x0[keep], ylo[keep], yhi[keep])
    assert not r["ok"]
    # a first-layer hit outside the loose window (Table 2: 0.8333 + 3.3333/5 = 1.5 mm) is not used
    x0b = x0.copy(); x0b[tidx[0]] += 1.6
    r = oracle64.ut_search(velo, qop, off, x0b, ylo, yhi)
    assert r["idx"][0] == NO_HIT and r["n"] == 3
    x0b[tidx[0]] = x0[tidx[0]] + 1.4
    r = oracle64.ut_search(velo, qop, off, x0b, ylo, yhi)
    assert r["idx"][0] == tidx[0]
    # a hit whose strip does not cover the predicted y (beyond the 1 mm tolerance) is ignored
    ylo_b, yhi_b = ylo.copy(), yhi.copy(); ylo_b[tidx[1]] += 300; yhi_b[tidx[1]] += 300
    r = oracle64.ut_search(velo, qop, off, x0, ylo_b, yhi_b)
    assert r["idx"][1] == NO_HIT and r["n"] == 3


def test_ut_strip_coverage_and_window_edges(oracle64):
    """O13 in numbers (L305-311, Table 2, reading A18).  (a) A hit inside the LOOSE window whose strip does not
    cover the predicted y (beyond the 1 mm tolerance) starts no hypothesis, on either side of the strip; one that
    misses y by less than the tolerance does.  (b) A hit outside a TIGHT window is never attached, even when it
    is the only hit of its layer."""
    qop = 1 / 5000.0
    gamma = AG + BG * qop
    velo = [1.0, -2.0, 0.05, 0.02]                       # y at UTaX: -2 + 0.02 * 1557 = 29.14 mm, strip row [0, 100]
    off, x0, ylo, yhi, tidx = make_ut(velo, gamma)
    y0 = velo[1] + velo[3] * (UT_Z[0] - 770.0)
    # (a) first layer: strip moved above / below the predicted y by more than the tolerance -> not used
    for lo_, hi_ in ((y0 + 1.5, y0 + 101.5), (y0 - 101.5, y0 - 1.5)):
        ylo_b, yhi_b = ylo.copy(), yhi.copy(); ylo_b[tidx[0]], yhi_b[tidx[0]] = lo_, hi_
        r = oracle64.ut_search(velo, qop, off, x0, ylo_b, yhi_b)
        assert r["idx"][0] == NO_HIT and r["n"] == 3, (lo_, hi_)
    # ... by less than the tolerance -> used
    for lo_, hi_ in ((y0 + 0.5, y0 + 100.5), (y0 - 100.5, y0 - 0.5)):
        ylo_b, yhi_b = ylo.copy(), yhi.copy(); ylo_b[tidx[0]], yhi_b[tidx[0]] = lo_, hi_
        r = oracle64.ut_search(velo, qop, off, x0, ylo_b, yhi_b)
        assert r["idx"][0] == tidx[0] and r["n"] == 4, (lo_, hi_)
    # the same for a tight-window layer
    y2 = velo[1] + velo[3] * (UT_Z[2] - 770.0)
    for lo_, hi_, used in ((y2 + 1.5, y2 + 101.5, False), (y2 - 101.5, y2 - 1.5, False), (y2 + 0.5, y2 + 100.5, True),
                           (y2 - 100.5, y2 - 0.5, True)):
        ylo_b, yhi_b = ylo.copy(), yhi.copy(); ylo_b[tidx[2]], yhi_b[tidx[2]] = lo_, hi_
        r = oracle64.ut_search(velo, qop, off, x0, ylo_b, yhi_b)
        assert (r["idx"][2] == tidx[2]) == used and r["n"] == (4 if used else 3), (lo_, hi_)
    # (b) tight windows at p = 5 GeV (Table 2): UTaU 0.2 + 0.6/5 -> 0.5 mm (lower clamp), UTbV 0.4 + 1.2/5 = 0.64 -> 1.0 mm
    for layer, inside, outside in ((1, 0.45, 0.55), (2, 0.95, 1.05), (3, 0.95, 1.05)):
        for sgn in (+1.0, -1.0):
            x0b = x0.copy(); x0b[tidx[layer]] += sgn * outside
            r = oracle64.ut_search(velo, qop, off, x0b, ylo, yhi)
            assert r["idx"][layer] == NO_HIT and r["n"] == 3, (layer, sgn)
            x0b = x0.copy(); x0b[tidx[layer]] += sgn * inside
            r = oracle64.ut_search(velo, qop, off, x0b, ylo, yhi)
            assert r["idx"][layer] == tidx[layer] and r["n"] == 4, (layer, sgn)


def test_ut_best_hypothesis_is_max_hits_then_min_residuals_then_first(oracle64):
    """Reading A13 (L309 "one or more UT hits"): every loose-window hit of the first layer with hits starts a
    hypothesis; the best has the most hits, then the smallest sum of squared residuals, then the lowest first hit.
    A decoy 0.3 mm beside the true first-layer hit also collects four hits (the tight windows still hold the true
    hits) but with residuals: the true hit must win whether it comes before or after the decoy."""
    qop = 1 / 5000.0
    gamma = AG + BG * qop
    velo = [1.0, -2.0, 0.05, 0.02]
    for d in (+0.3, -0.3):
        off, x0, ylo, yhi, tidx = make_ut(velo, gamma, extra=[(0, d)])
        decoy = int(tidx[0]) + (1 if d > 0 else -1)
        assert off[1] == 2 and x0[decoy] == pytest.approx(x0[tidx[0]] + d)
        r = oracle64.ut_search(velo, qop, off, x0, ylo, yhi)
        assert r["ok"] and r["n"] == 4 and (r["idx"] == tidx).all(), d
        assert r["ssq"] < 1e-16 and r["gamma"] == pytest.approx(gamma, rel=1e-9)
        # alone, the decoy's hypothesis has four hits too, with a visible sum of squared residuals
        keep = np.ones(len(x0), bool); keep[tidx[0]] = False
        off1 = off.copy(); off1[1:] -= 1
        r1 = oracle64.ut_search(velo, qop, off1, x0[keep], ylo[keep], yhi[keep])
        assert r1["ok"] and r1["n"] == 4 and r1["ssq"] > 1e-3
        # the sum of squared residuals is what its name says (Eq. 19 with the refitted gamma_x)
        xs, ys = x0[keep], None
        res = []
        for i in range(4):
            j = r1["idx"][i]; dz = UT_Z[i] - 770.0
            yy = velo[1] + velo[3] * dz
            res.append((xs[j] + yy * UT_TAN[i]) - (velo[0] + velo[2] * dz + r1["gamma"] * dz * dz))
        assert r1["ssq"] == pytest.approx(float(np.sum(np.square(res))), rel=1e-9)
    # more hits beat smaller residuals: the true first-layer hit with its layer-2 and layer-3 hits removed
    # (two hits) loses against ... nothing: fewer than three hits is no candidate; with layer 3 only removed the
    # three-hit true hypothesis still beats a far decoy that reaches one hit
    off, x0, ylo, yhi, tidx = make_ut(velo, gamma, extra=[(0, 1.2)])
    keep = np.ones(len(x0), bool); keep[tidx[3] ] = False
    off2 = off.copy(); off2[4:] -= 1
    r = oracle64.ut_search(velo, qop, off2, x0[keep], ylo[keep], yhi[keep])
    assert r["ok"] and r["n"] == 3 and r["idx"][0] == tidx[0] and r["idx"][3] == NO_HIT
    # exact duplicates of the first-layer hit: identical hypotheses, the lower index stays
    off, x0, ylo, yhi, tidx = make_ut(velo, gamma, extra=[(0, 0.0)])
    r = oracle64.ut_search(velo, qop, off, x0, ylo, yhi)
    assert r["n"] == 4 and r["idx"][0] == 0 and x0[0] == x0[1]


def test_refined_qop_is_eq20_inverted(geom):
    """L307 / Eq. 20: the long track's q/p comes from the refitted gamma_x, q/p = (gamma_x - A_gamma) / B_gamma
    (times the polarity).  One seed, one VELO state, four noise-free UT hits of a 6 GeV track: the output q/p is
    the truth to 1e-6 (A_gamma alone is 5e-5 of gamma_x here), whereas the kick estimate it starts from is 2% off."""
    from types import SimpleNamespace
    for mode, pol in (("f64", -1), ("f64", +1)):
        o = Oracle(geom, mode)
        q_true = 1.0 / 6000.0
        gamma = AG + BG * q_true
        velo = [1.0, -2.0, 0.05, 0.02]
        off, x0, ylo, yhi, tidx = make_ut(velo, gamma)
        dtx = q_true * geom["kick_pt"] * 1.02                 # the kick estimate (A10): 2% off
        txs = velo[2] + dtx
        seed = [0.0, velo[1] + velo[3] * (7826.0 - 770.0), txs, velo[3], 0.0]
        for _ in range(6):
            zm = o.match_pair(seed[:4], velo)["zm"]
            seed[0] = (velo[0] + (zm - 770.0) * velo[2]) - (zm - 7826.0) * txs
        ev = SimpleNamespace(n_events=1, polarity=np.array([pol], np.int8), velo_off=np.array([0, 1], np.uint32),
                             velo_x=np.array([velo[0]]), velo_y=np.array([velo[1]]), velo_tx=np.array([velo[2]]),
                             velo_ty=np.array([velo[3]]), ut_off=off, ut_x0=x0, ut_ylo=ylo, ut_yhi=yhi)
        m = o.matching(1, np.array([0, 1], np.uint32), np.array([seed]), ev, use_ut=True)
        assert m["n"] == 1 and m["n_ut"][0] == 4
        assert m["qop"][0] == pytest.approx(pol * q_true, rel=1e-6)
        m0 = o.matching(1, np.array([0, 1], np.uint32), np.array([seed]), ev, use_ut=False)
        assert m0["qop"][0] == pytest.approx(pol * q_true * 1.02, rel=1e-9)


def test_selection_is_one_to_one(geom):
    ev = generate(config(5, 40))
    for mode in ("f32", "f64"):
        o = Oracle(geom, mode)
        m = o.matching(ev.n_events, ev.seed_off, ev.seed_state.T, ev)
        assert m["n"] > 40 * 100
        assert len(np.unique(m["seed"])) == m["n"] and len(np.unique(m["velo"])) == m["n"]
        assert (m["chi2"] < 2.0).all() and (m["n_ut"] >= 3).all()
        for i in range(m["n"]):        # pair belongs to one event; UT hits in that event's layers
            e = m["event"][i]
            assert ev.seed_off[e] <= m["seed"][i] < ev.seed_off[e + 1]
            assert ev.velo_off[e] <= m["velo"][i] < ev.velo_off[e + 1]
            for l in range(4):
                if m["ut"][i, l] != NO_HIT:
                    assert ev.ut_off[e * 4 + l] <= m["ut"][i, l] < ev.ut_off[e * 4 + l + 1]
        good = ev.seed_pid[m["seed"]] == ev.velo_pid[m["velo"]]
        assert good.mean() > 0.97
        # efficiency on true partners whose UT hits exist
        P = ev.particles
        den = (ev.seed_pid >= 0) & (P["n_ut"][np.maximum(ev.seed_pid, 0)] >= 3)
        found = np.zeros(len(ev.seed_pid), bool); found[m["seed"][good]] = True
        assert found[den].mean() > 0.85
        # refined q/p close to truth for correct matches
        t_qop = (P["q"] / P["p"])[ev.seed_pid[m["seed"][good]]]
        rel = np.abs(m["qop"][good] / t_qop - 1)
        assert np.median(rel) < 0.02


def test_matching_without_ut_keeps_more(geom):
    ev = generate(config(5, 10))
    o = Oracle(geom, "f32")
    with_ut = o.matching(ev.n_events, ev.seed_off, ev.seed_state.T, ev, use_ut=True)
    no_ut = o.matching(ev.n_events, ev.seed_off, ev.seed_state.T, ev, use_ut=False)
    assert no_ut["n"] >= with_ut["n"] and (no_ut["n_ut"] == 0).all()
    # kick estimate of q/p (A10) has the right sign and size
    good = ev.seed_pid[no_ut["seed"]] == ev.velo_pid[no_ut["velo"]]
    P = ev.particles
    t = (P["q"] / P["p"])[ev.seed_pid[no_ut["seed"][good]]]
    assert np.median(np.abs(no_ut["qop"][good] / t - 1)) < 0.05


def test_full_chain_cfg2(cfg2_small, oracle32):
    ev = cfg2_small
    s, m = oracle32.reconstruct(ev)
    pid, _ = truth.seed_pids(ev, s["hits"])
    summ = truth.long_summary(ev, pid[m["seed"]], m["velo"])
    assert summ["efficiency"] > 0.9 and summ["ghost_rate"] < 0.02
    assert len(np.unique(m["seed"])) == m["n"] and len(np.unique(m["velo"])) == m["n"]
