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
