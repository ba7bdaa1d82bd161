"""Pins of the oracle's seeding steps O2..O10: brute force, textbook special cases, library
least squares, noise-free recovery from the paper's track model, clone-kill worked examples and
invariants (SURVEY.md 8(c) "What pins each part")."""
import itertools
from dataclasses import replace

import numpy as np
import pytest

from lhcb_gen import config, default_geom, generate, truth, X_LAYERS, UV_LAYERS
from oracle.binding import Oracle, NO_HIT

Z = np.array(default_geom()["scifi_z"])
ZREF = 8525.0
DR = -3.3e-4


def g_of(z, d=DR):
    zb = z - ZREF
    return zb * zb * (1 + d * zb)


# ----------------------------------------------------------------------------- O2-O4 brute force
def brute_triplets(ev, geom, event, half):
    """All (it, i1, i2, i3) that the paper's cuts accept, by exhaustive enumeration in float64 with
    the equations in their printed form: Eq. 11 window; Eq. 3-5 momentum; c_x solved from the
    three points with a 3x3 linear system and compared to the (1/p, s*c_x) band.
    Returns (accepted set, set of triples within 1e-3 relative of any cut edge)."""
    a, b = geom["inv_p_a"], geom["inv_p_b"]
    f_lo, f_hi, d_lo, d_hi = geom["cx_band"]
    out, edge = set(), set()
    base = (event * 2 + half) * 12
    x = ev.hit_x.astype(np.float64)
    for it, (l1, l2, l3) in enumerate(geom["iter_layers"]):
        z1, z2, z3 = Z[l1], Z[l2], Z[l3]
        dx3 = (z3 - z1) / (2 * z1 * b) * (-a + np.sqrt(a * a + 4 * b / geom["p_min"]))
        acorr = geom["alpha0"] / (z1 / (z3 - z1) * (geom["p_min"] - geom["alpha1"]))
        M = np.array([[1, z - ZREF, g_of(z)] for z in (z1, z2, z3)])
        Minv2 = np.linalg.inv(M)[2]      # c_x row of the 3-point solution (library inverse)
        r1 = range(ev.zone_off[base + l1], ev.zone_off[base + l1 + 1])
        r2 = range(ev.zone_off[base + l2], ev.zone_off[base + l2 + 1])
        r3 = range(ev.zone_off[base + l3], ev.zone_off[base + l3 + 1])
        for i1, i3 in itertools.product(r1, r3):
            c = (z3 + acorr) / z1 * x[i1]
            u = abs(x[i3] - c) / dx3
            if u > 1 + 1e-6:
                continue
            near13 = abs(u - 1) < 1e-6
            t13 = (x[i3] - x[i1]) / (z3 - z1)
            x0 = x[i1] - z1 * t13
            s = 1.0 if x0 >= 0 else -1.0
            invp = a * abs(x0) + b * x0 * x0
            cxp = -s * geom["kappa_cx"] * invp
            lo = min(f_lo * cxp, f_hi * cxp) - d_lo
            hi = max(f_lo * cxp, f_hi * cxp) + d_hi
            tol = 2e-10          # ~1e-4 mm at the T2 layer: float32 rounding of the window edges
            i2s = np.arange(r2.start, r2.stop)
            cxs = Minv2[0] * x[i1] + Minv2[1] * x[i2s] + Minv2[2] * x[i3]
            for i2, cx in zip(i2s[(cxs >= lo - tol) & (cxs <= hi + tol)], cxs[(cxs >= lo - tol) & (cxs <= hi + tol)]):
                inside = lo + tol <= cx <= hi - tol and u < 1 - 1e-6
                (out if inside and not near13 else edge).add((it, i1, int(i2), i3))
    return out, edge


@pytest.mark.parametrize("cfgname", ["cfg1", "cfg2"])
def test_triplets_equal_brute_force(cfgname, oracle32, cfg1_events, cfg2_small, geom):
    ev = cfg1_events if cfgname == "cfg1" else cfg2_small
    n_ev = 16 if cfgname == "cfg1" else 2
    total = 0
    for event in range(n_ev):
        for half in (0, 1):
            d = oracle32.seeding_debug(ev, event, half)
            got = {(int(i), *map(int, t)) for i, t in zip(d["t_it"], d["t_idx"][:, [0, 1, 2]])}
            sure, edge = brute_triplets(ev, geom, event, half)
            assert sure <= got, "oracle misses triplets the cuts accept"
            assert got <= (sure | edge), "oracle accepts triplets outside the cuts"
            total += len(got)
    assert total > 500


def test_triplets_equal_brute_force_with_an_asymmetric_band(cfg2_small):
    """PAPER.md L175 ("one side exhibits a longer tail"; reading A4): the additive widths of the c_x band differ on
    its two sides.  The default geometry has d_lo = d_hi, which hides a swap; here d_lo = 0.5e-6, d_hi = 2e-6."""
    from lhcb_gen import default_geom
    from oracle.binding import Oracle
    g = default_geom(cx_band=[0.5, 1.8, 0.5e-6, 2.0e-6])
    o = Oracle(g, "f32")
    ev = cfg2_small
    total = n_sym = 0
    for event in range(2):
        for half in (0, 1):
            d = o.seeding_debug(ev, event, half)
            got = {(int(i), *map(int, t)) for i, t in zip(d["t_it"], d["t_idx"][:, [0, 1, 2]])}
            sure, edge = brute_triplets(ev, g, event, half)
            assert sure <= got, "oracle misses triplets the cuts accept"
            assert got <= (sure | edge), "oracle accepts triplets outside the cuts"
            # the same cuts with the two widths swapped accept a different set: the asymmetry is exercised
            swapped, _ = brute_triplets(ev, dict(g, cx_band=[0.5, 1.8, 2.0e-6, 0.5e-6]), event, half)
            n_sym += len(sure ^ swapped)
            total += len(got)
    assert total > 500 and n_sym > 50


# ----------------------------------------------------------------------------- O5 exact parabola
def test_parabola3_is_lagrange_when_dratio_zero():
    g = default_geom(d_ratio=0.0)
    o = Oracle(g, "f64")
    rng = np.random.default_rng(5)
    for it, (l1, l2, l3) in enumerate(g["iter_layers"]):
        zb = Z[[l1, l2, l3]] - ZREF
        for _ in range(20):
            xs = rng.uniform(-2000, 2000, 3)
            c2, c1, c0 = np.polyfit(zb, xs, 2)          # textbook quadratic interpolation
            ax, bx, cx = o.parabola3(it, *xs)
            assert ax == pytest.approx(c0, rel=1e-9, abs=1e-7)
            assert bx == pytest.approx(c1, rel=1e-9, abs=1e-11)
            assert cx == pytest.approx(c2, rel=1e-8, abs=1e-13)


def test_parabola3_passes_through_hits(oracle64):
    rng = np.random.default_rng(6)
    for it, (l1, l2, l3) in enumerate(default_geom()["iter_layers"]):
        for _ in range(20):
            xs = rng.uniform(-2000, 2000, 3)
            ax, bx, cx = oracle64.parabola3(it, *xs)
            for z, x in zip(Z[[l1, l2, l3]], xs):
                assert ax + bx * (z - ZREF) + cx * g_of(z) == pytest.approx(x, abs=1e-8)


# ----------------------------------------------------------------------------- O6 / O9 fits
@pytest.mark.parametrize("missing", [-1, 0, 1, 2, 3, 4, 5])
def test_fit_xz_equals_lstsq(missing, oracle64, geom):
    rng = np.random.default_rng(7 + missing)
    zx = Z[X_LAYERS]
    A = np.stack([np.ones(6), zx - ZREF, g_of(zx)], 1)
    for it in (0, 1):
        seeds = {X_LAYERS.index(l) for l in geom["iter_layers"][it]}
        if missing in seeds:
            continue
        for _ in range(10):
            truth_par = np.array([rng.uniform(-2000, 2000), rng.uniform(-0.5, 0.5), rng.uniform(-1e-5, 1e-5)])
            xs = A @ truth_par + rng.normal(0, 0.08, 6)
            keep = [s for s in range(6) if s != missing]
            sol, res, *_ = np.linalg.lstsq(A[keep], xs[keep], rcond=None)
            ax, bx, cx, chi2 = oracle64.fit_xz(it, xs, missing)
            assert ax == pytest.approx(sol[0], rel=1e-9, abs=1e-8)
            assert bx == pytest.approx(sol[1], rel=1e-9, abs=1e-12)
            assert cx == pytest.approx(sol[2], rel=1e-7, abs=1e-14)
            r = xs[keep] - A[keep] @ sol
            assert chi2 == pytest.approx((r @ r) / 0.08 ** 2 / (len(keep) - 3), rel=1e-6)
    # the f32 build applies the same map: agrees with lstsq to float accuracy
    o32 = Oracle(geom, "f32")
    xs = (A @ np.array([812.0, 0.21, 3e-6]) + rng.normal(0, 0.08, 6)).astype(np.float32).astype(np.float64)
    keep = [s for s in range(6) if s != missing]
    it = 0 if missing not in {0, 2, 4} else 1
    sol, *_ = np.linalg.lstsq(A[keep], xs[keep], rcond=None)
    ax, bx, cx, chi2 = o32.fit_xz(it, xs, missing)
    assert ax == pytest.approx(sol[0], abs=5e-3) and bx == pytest.approx(sol[1], abs=1e-6)
    assert cx == pytest.approx(sol[2], abs=1e-9)


def test_fit_y_equals_lstsq(oracle64, geom):
    rng = np.random.default_rng(11)
    zu = Z[UV_LAYERS]
    ta = np.array(geom["scifi_tan_alpha"])[UV_LAYERS]
    for mask in [m for m in range(64) if bin(m).count("1") >= 4]:
        keep = [s for s in range(6) if mask >> s & 1]
        ay, by = rng.uniform(-2000, 2000), rng.uniform(-0.3, 0.3)
        y = ay + by * (zu - ZREF)
        m = -y * ta + rng.normal(0, 0.08, 6)        # x_hit - x_pred = -y tan(alpha) + noise
        A = np.stack([ta, ta * (zu - ZREF)], 1)
        sol, *_ = np.linalg.lstsq(A[keep], -m[keep], rcond=None)
        g_ay, g_by, chi2 = oracle64.fit_y(mask, m)
        assert g_ay == pytest.approx(sol[0], rel=1e-9, abs=1e-7)
        assert g_by == pytest.approx(sol[1], rel=1e-9, abs=1e-10)
        r = m[keep] + A[keep] @ sol
        assert chi2 == pytest.approx((r @ r) / 0.08 ** 2 / (len(keep) - 2), rel=1e-6, abs=1e-12)


# ----------------------------------------------------------------------------- noise-free recovery
def test_noise_free_tracks_recovered_exactly(geom):
    """Tracks generated exactly from the paper's track model (Eq. 1, straight y) with no noise:
    100% of reconstructible tracks found, fit parameters equal truth to 1e-6 relative (f64)."""
    cfg = replace(config(1), sigma_x=0.0, n_events=32, seed=123)
    ev = generate(cfg)
    o = Oracle(geom, "f64")
    s = o.seeding(ev)
    pid, pur = truth.seed_pids(ev, s["hits"])
    assert (pid >= 0).all() and (pur == 1.0).all()
    den = truth.reconstructible_seed(ev)
    found = np.zeros(len(den), bool); found[pid] = True
    assert den.sum() > 500 and found[den].all()
    P = ev.particles
    for k, name in enumerate(["ax", "bx", "cx", "ay", "by"]):
        t = P[name][pid]; got = s["par"][:, k]
        floor = {"ax": 1e-3, "bx": 1e-6, "cx": 1e-9, "ay": 1e-3, "by": 1e-6}[name]
        assert np.all(np.abs(got - t) <= 1e-6 * np.maximum(np.abs(t), floor)), name
    assert (s["par"][:, 5] < 1e-12).all() and (s["par"][:, 6] < 1e-12).all()
    # state at z_S: x, y, tx, ty, q/p
    assert np.allclose(s["state"][:, 0], P["x_S"][pid], rtol=1e-9, atol=1e-7)
    assert np.allclose(s["state"][:, 2], P["tx_S"][pid], rtol=1e-7, atol=1e-10)
    assert np.allclose(s["state"][:, 4], (P["q"] / P["p"])[pid], rtol=1e-5)
    # each found track has all its hits (12) and every track is found once
    assert ((s["nx"] == 6) & (s["nuv"] == 6))[den[pid]].all()
    assert len(np.unique(pid)) == len(pid)


def test_f32_and_f64_oracles_agree_on_cfg1(cfg1_events, oracle32, oracle64):
    a, b = oracle32.seeding(cfg1_events), oracle64.seeding(cfg1_events)
    sa = {tuple(h) for h in a["hits"]}; sb = {tuple(h) for h in b["hits"]}
    assert len(sa ^ sb) <= 0.01 * len(sa)


# ----------------------------------------------------------------------------- O7 clone kill
def hits6(*idx):
    return list(idx) + [NO_HIT] * (6 - len(idx))


def test_clone_kill_worked_examples(oracle32):
    """SURVEY.md 8(c), derived from PAPER.md L189-198.  A: six hits, chi2 0.5 -> score 500."""
    k = oracle32.clone_key
    A = hits6(0, 1, 2, 3, 4, 5)
    # 1. B: five hits, shares 3 with A, chi2 0.02 -> score 200.  B owns 5, A owns 3: both kept.
    keep = oracle32.clone_kill([k(0.5, 1e-6, 6), k(0.02, 1e-6, 5)], [A, hits6(0, 1, 2, 6, 7)], [6, 5], 8)
    assert keep.tolist() == [True, True]
    # 2. B shares 4: A owns 2 and has six hits: both kept.
    keep = oracle32.clone_kill([k(0.5, 1e-6, 6), k(0.02, 1e-6, 5)], [A, hits6(0, 1, 2, 3, 6)], [6, 5], 7)
    assert keep.tolist() == [True, True]
    # 3. B chi2 0.06 -> score 600 > 500.  A owns 6, B owns 1: B dropped.
    keep = oracle32.clone_kill([k(0.5, 1e-6, 6), k(0.06, 1e-6, 5)], [A, hits6(0, 1, 2, 3, 6)], [6, 5], 7)
    assert keep.tolist() == [True, False]
    # a five-hit track wins only if its chi2 is more than ten times smaller (L192)
    assert k(0.049, 0, 5) < k(0.5, 0, 6) < k(0.051, 0, 5)
    # c_x tie-break prefers higher momentum = smaller |c_x| (L192); iteration breaks exact ties
    assert k(0.5, 1e-6, 6) < k(0.5, -2e-6, 6)
    assert k(0.5, 1e-6, 6, 0) < k(0.5, 1e-6, 6, 1)
    # a five-hit track that keeps only two of its hits is dropped, a six-hit one is kept (L198)
    keep = oracle32.clone_kill([k(0.1, 0, 6), k(0.2, 0, 5)], [A, hits6(0, 1, 2, 6, 7)], [6, 5], 8)
    assert keep.tolist() == [True, False]
    keep = oracle32.clone_kill([k(0.1, 0, 6), k(0.2, 0, 6)], [A, hits6(0, 1, 2, 3, 6, 7)], [6, 6], 8)
    assert keep.tolist() == [True, True]
    # a five-hit track that keeps exactly three of its hits is retained ("at least three", L198), with four too
    keep = oracle32.clone_kill([k(0.1, 0, 6), k(0.2, 0, 5)], [A, hits6(0, 1, 6, 7, 8)], [6, 5], 9)
    assert keep.tolist() == [True, True]
    keep = oracle32.clone_kill([k(0.1, 0, 6), k(0.2, 0, 5)], [A, hits6(0, 6, 7, 8, 9)], [6, 5], 10)
    assert keep.tolist() == [True, True]
    # a six-hit track that keeps one hit only is dropped (two are needed, L198)
    keep = oracle32.clone_kill([k(0.1, 0, 6), k(0.2, 0, 6)], [A, hits6(0, 1, 2, 3, 4, 6)], [6, 6], 7)
    assert keep.tolist() == [True, False]


def test_clone_kill_invariants(oracle32, cfg2_small):
    rng = np.random.default_rng(3)
    d = oracle32.seeding_debug(cfg2_small, 0, 0)
    n = len(d["c_key"])
    assert n > 50
    base = int(cfg2_small.zone_off[0]); nh = int(cfg2_small.zone_off[12]) - base
    hits = np.where(d["c_hits"] == NO_HIT, NO_HIT, d["c_hits"] - base).astype(np.uint32)
    keep = oracle32.clone_kill(d["c_key"], hits, d["c_nx"], nh)
    assert (keep == d["c_keep"].astype(bool)).all()
    # order independence
    perm = rng.permutation(n)
    keep_p = oracle32.clone_kill(d["c_key"][perm], hits[perm], d["c_nx"][perm], nh)
    assert (keep_p == keep[perm]).all()
    # candidates on disjoint hits all survive
    dis = np.arange(60, dtype=np.uint32).reshape(10, 6)
    assert oracle32.clone_kill(rng.integers(1, 2 ** 40, 10).astype(np.uint64), dis, [6] * 10, 60).all()
    # an exact duplicate with the worse key dies
    keep2 = oracle32.clone_kill([5, 9], [hits6(*range(6))] * 2, [6, 6], 6)
    assert keep2.tolist() == [True, False]
    # clone fraction before/after: duplicates of a kept candidate's hit set do not survive
    kept_sets = [tuple(h) for h in d["c_hits"][keep]]
    assert len(set(kept_sets)) == len(kept_sets)
    assert 0.3 < 1 - keep.mean() < 0.8          # about half of the candidates are clones (L185)


# ----------------------------------------------------------------------------- O8-O10 invariants
@pytest.mark.parametrize("mode", ["f32", "f64"])
def test_seed_invariants(mode, cfg2_small, geom):
    o = Oracle(geom, mode)
    ev = cfg2_small
    s = o.seeding(ev)
    hits = s["hits"]
    assert s["n"] > 100 * ev.n_events / 2
    x = (ev.hit_x if mode == "f32" else ev.hit_x64).astype(np.float64)
    ta = np.array(geom["scifi_tan_alpha"])
    for i in range(s["n"]):
        h = hits[i]
        zbase = (s["event"][i] * 2 + s["half"][i]) * 12
        for l in range(12):       # at most one hit per layer, and it lies in this half's zone of that layer
            if h[l] != NO_HIT:
                assert ev.zone_off[zbase + l] <= h[l] < ev.zone_off[zbase + l + 1]
        nx = sum(h[l] != NO_HIT for l in X_LAYERS); nuv = sum(h[l] != NO_HIT for l in UV_LAYERS)
        assert nx == s["nx"][i] and nuv == s["nuv"][i]
        assert nx in (5, 6) and nuv in (4, 5, 6)
        ax, bx, cx, ay, by, c2x, c2y = s["par"][i].astype(np.float64)
        assert c2x <= 8.0 and c2y <= 8.0
        for l in range(12):       # residuals of the attached hits w.r.t. the final fit are small
            if h[l] == NO_HIT:
                continue
            zb = Z[l] - ZREF
            pred = ax + bx * zb + cx * g_of(Z[l]) - (ay + by * zb) * ta[l]
            assert abs(x[h[l]] - pred) < (1.0 if ta[l] == 0 else 2.0) + 1e-3
    # a hit is used by at most a handful of seeds and no two seeds are identical
    sets = [tuple(h) for h in hits]
    assert len(set(sets)) == len(sets)
    summ = truth.seeding_summary(ev, hits)
    assert summ["efficiency"] > 0.95 and summ["ghost_rate"] < 0.02 and summ["clone_rate"] < 0.02


def test_window_containment_of_toy_model(geom, oracle64):
    """Generator self-test: every in-acceptance track with p >= 1.15 p_min has its
    T3 hit inside the Eq. 11 window and its T2 hit inside the third-hit band."""
    cfg = replace(config(1), sigma_x=0.0, n_events=200, seed=77, p_lo=3450.0)
    ev = generate(cfg)
    P = ev.particles
    c = oracle64.constants()
    worst13 = 0.0
    for it, (l1, l2, l3) in enumerate(geom["iter_layers"]):
        x1, x2, x3 = (P["ax"] + P["bx"] * (Z[l] - ZREF) + P["cx"] * g_of(Z[l]) for l in (l1, l2, l3))
        ok = P["in_acc"]
        u = np.abs(x3 - c["r13"][it] * x1) / c["dx3max"][it]
        worst13 = max(worst13, u[ok].max())
        for i in np.nonzero(ok)[0][:300]:
            m = oracle64.momentum(it, x1[i], x3[i])
            assert m["lo2"] <= x2[i] <= m["hi2"]
    assert worst13 < 1.0
