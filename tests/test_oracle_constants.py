"""Pins of the oracle's closed-form pieces against values fixed by the paper's printed constants
(tests/golden/closed_forms.txt; none produced by code in this repository)."""
import math
import os

import numpy as np
import pytest

from lhcb_gen import default_geom
from oracle.binding import Oracle

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")) as f:
    for line in f:
        if line.strip() and not line.startswith("#"):
            name, val, tol = line.split()[:3]
            GOLD[name] = (float(val), float(tol))


def check(name, got):
    want, tol = GOLD[name]
    assert got == pytest.approx(want, rel=tol), (name, got, want)


@pytest.mark.parametrize("mode", ["f32", "f64"])
def test_window_constants(mode, geom):
    o = Oracle(geom, mode)
    c = o.constants()
    check("dx3max_it0", c["dx3max"][0]); check("dx3max_it1", c["dx3max"][1])
    check("alpha_corr_it0", c["alpha_corr"][0]); check("alpha_corr_it1", c["alpha_corr"][1])
    check("K_it0", c["K"][0]); check("K_it1", c["K"][1])
    # Eq. 7: dx3max = (z3 - z1)/z1 * x0_max  -> x0_max, "independent from the choice of layers" (L133)
    z = geom["scifi_z"]
    for it, (l1, _, l3) in enumerate(geom["iter_layers"]):
        check("x0_max_pmin3000", c["dx3max"][it] * z[l1] / (z[l3] - z[l1]))
    # Eq. 11: window centre factor (z3 + alpha_corr)/z1
    assert c["r13"][0] == pytest.approx((9193 + 93.491) / 7826, rel=2e-6)


def test_invp_at_x0max_is_pmin(oracle64, geom):
    """Eq. 5 evaluated by the oracle at the Eq. 8 root returns 1/p_min (x3 chosen so that x0 = 2189.76)."""
    z1, z3 = 7826.0, 9193.0
    x0 = GOLD["x0_max_pmin3000"][0]
    x1 = 100.0
    t13 = (x1 - x0) / z1
    m = oracle64.momentum(0, x1, x1 + t13 * (z3 - z1))
    assert m["x0"] == pytest.approx(x0, rel=1e-9)
    assert 1.0 / m["invp"] == pytest.approx(3000.0, rel=5e-6)
    assert m["s"] == 1.0
    m = oracle64.momentum(0, -x1, -(x1 + t13 * (z3 - z1)))
    assert m["s"] == -1.0 and 1.0 / m["invp"] == pytest.approx(3000.0, rel=5e-6)


def test_pmin_domain():
    lim = GOLD["pmin_domain"][0]
    ok = Oracle(default_geom(p_min=lim * 1.001), "f64").constants()["dx3max"]
    bad = Oracle(default_geom(p_min=lim * 0.999), "f64").constants()["dx3max"]
    assert np.isfinite(ok).all() and np.isnan(bad).all()


def test_K_is_chord_sagitta_without_dratio():
    """A3: with d_ratio = 0, K = (z2 - z1)(z2 - z3) (textbook sagitta of a parabola under its chord)."""
    g = default_geom(d_ratio=0.0)
    K = Oracle(g, "f64").constants()["K"]
    z = g["scifi_z"]
    for it, (l1, l2, l3) in enumerate(g["iter_layers"]):
        assert K[it] == pytest.approx((z[l2] - z[l1]) * (z[l2] - z[l3]), rel=1e-13)


@pytest.mark.parametrize("mode,rel", [("f32", 2e-6), ("f64", 1e-9)])
def test_zmatch_and_tolerances(mode, rel, geom):
    o = Oracle(geom, mode)
    # z_match depends on |dtx|, |x_S| and tx_V only: dtx = tx_S - tx_V
    for name, dtx, x, tx in (("zmatch_0_0_0", 0.0, 0.0, 0.0), ("zmatch_0.4_1500_0.25", 0.4, 1500.0, 0.25),
                             ("zmatch_0.04_500_0.1", 0.04, 500.0, 0.1)):
        for sx in (1, -1):
            for sd in (1, -1):
                r = o.match_pair([sx * x, 0.0, tx + sd * dtx, 0.0], [0.0, 0.0, tx, 0.0])
                check(name, r["zm"])
    # Eq. 22-23: isolate each term of chi2 with the others zero
    # (a) dtx = 0.1, dx = dy = dty = 0 is not reachable exactly, so use the identity
    #     chi2 = dx^2/tolx + dtx^2/0.5 and solve for tolx from the reported dx, chi2
    sd = [10.0, 0.0, 0.1, 0.0]; vl = [0.0, 0.0, 0.0, 0.0]
    r = o.match_pair(sd, vl)
    # y part: y_S + (10000-7826)*0 - 0 = 0 ; dty = 0
    tolx = r["dx"] ** 2 / (r["chi2"] - r["dtx"] ** 2 / 0.5)
    assert r["presel"] == 0 or tolx == pytest.approx(GOLD["tolx_dtx0.1"][0], rel=1e-3)
    # choose x_S so that dx is small enough to pass preselection
    zm = r["zm"]
    xs = -(zm - 7826.0) * 0.1 + 5.0          # then dx ~ 5 mm
    r = o.match_pair([xs, 0.0, 0.1, 0.0], vl)
    assert r["presel"] == 1.0
    tolx = r["dx"] ** 2 / (r["chi2"] - r["dtx"] ** 2 / 0.5)
    assert tolx == pytest.approx(GOLD["tolx_dtx0.1"][0], rel=max(rel * 50, 1e-6))
    # (b) tol_y: dy only.  rho = tx_V^2 + ty_V^2
    for name, txv in (("toly_rho0", 0.0), ("toly_rho0.01", 0.1)):
        # collinear in x: seed on the VELO line (dtx = 0 -> z_m irrelevant), shifted by 0.5 mm in y
        xs = 0.0 + txv * (7826.0 - 770.0)
        r = o.match_pair([xs, 0.5, txv, 0.0], [0.0, 0.0, txv, 0.0])
        assert r["presel"] == 1.0 and abs(r["dx"]) < 1e-3 and r["dy"] == pytest.approx(0.5, rel=1e-6)
        toly = r["dy"] ** 2 / (r["chi2"] - r["dx"] ** 2 / 81.9)
        assert toly == pytest.approx(GOLD[name][0], rel=max(rel * 50, 1e-5))


def test_chi2_match_is_eq22_with_all_four_terms(oracle64):
    """Eq. 22-23 as printed, every term non-zero at once (t_y^VELO included in rho^VELO): the four terms are
    computed here from the pair's own dx, dy, dtx, dty and the printed constants."""
    for velo4, dtx, dty, dx_want, dy_want in (([3.0, -2.0, 0.045, -0.121], 0.036, 0.009, 7.0, -5.0),
                                              ([-1.5, 4.0, -0.070, 0.149], -0.028, -0.012, -11.0, 8.0)):
        xv, yv, txv, tyv = velo4
        txs, tys = txv + dtx, tyv + dty
        ys = (yv + (10000.0 - 770.0) * tyv) - (10000.0 - 7826.0) * tys + dy_want
        xs = 0.0
        for _ in range(6):                                   # z_match depends (weakly) on |x_S|: fixed point
            zm = oracle64.match_pair([xs, ys, txs, tys], velo4)["zm"]
            xs = (xv + (zm - 770.0) * txv) - (zm - 7826.0) * txs + dx_want
        seed4 = [xs, ys, txs, tys]
        r = oracle64.match_pair(seed4, velo4)
        txv, tyv = velo4[2], velo4[3]
        tolx = 0.8 * (10.12 ** 2 + 101.0 ** 2 * r["dtx"] ** 2)
        toly = 0.2 * (1.59 ** 2 + 212.1 ** 2 * (txv * txv + tyv * tyv))
        want = r["dx"] ** 2 / tolx + r["dy"] ** 2 / toly + r["dtx"] ** 2 / 0.5 + r["dty"] ** 2 * 937.5
        assert r["chi2"] == pytest.approx(want, rel=1e-12)
        # the slope terms and the t_y^VELO part of tol_y are visible at this size
        assert r["presel"] == 1.0 and abs(r["dx"] - dx_want) < 0.1 and abs(r["dy"] - dy_want) < 1e-6
        assert r["dty"] ** 2 * 937.5 > 0.05 * want and 212.1 ** 2 * tyv * tyv > 0.1 * 1.59 ** 2
        assert r["dty"] == pytest.approx(seed4[3] - velo4[3], rel=1e-12) and r["dtx"] == pytest.approx(seed4[2] - velo4[2], rel=1e-12)
        # dy is taken at z = 10 m: both lines extrapolated there (L231)
        assert r["dy"] == pytest.approx((seed4[1] + (10000.0 - 7826.0) * seed4[3]) - (velo4[1] + (10000.0 - 770.0) * velo4[3]), rel=1e-12)


def test_gamma_and_ut_windows(oracle64):
    check("gamma_qop_1over3000", oracle64.gamma(1.0 / 3000.0))
    check("deflection_UTaX_p3000", oracle64.gamma(1.0 / 3000.0) * (2327.0 - 770.0) ** 2)
    check("loose_UTaX_p3GeV", oracle64.ut_window(0, False, 1.0 / 3.0))
    check("loose_UTaX_p0.4GeV", oracle64.ut_window(0, False, 1.0 / 0.4))
    check("loose_UTaX_p100GeV", oracle64.ut_window(0, False, 1.0 / 100.0))
    # Table 2 tight rows: UTaU 0.2 + 0.6/p in [0.5, 2.0]; UTbV/UTbX 0.4 + 1.2/p in [1.0, 4.0]
    assert oracle64.ut_window(1, True, 1.0) == pytest.approx(0.8)
    assert oracle64.ut_window(1, True, 0.1) == pytest.approx(0.5)
    assert oracle64.ut_window(2, True, 1.0) == pytest.approx(1.6)
    assert oracle64.ut_window(3, True, 10.0) == pytest.approx(4.0)


def test_preselection_is_strict_and_field_off(oracle64):
    """Eq. 21 strict '<'; special case dtx = 0 and collinear segments: dx = 0, dy = 0, chi2 = 0."""
    tx, ty = 0.07, -0.03
    xs, ys = 1.0 + tx * (7826 - 770), 2.0 + ty * (7826 - 770)
    r = oracle64.match_pair([xs, ys, tx, ty], [1.0, 2.0, tx, ty])
    assert r["presel"] == 1 and abs(r["dx"]) < 1e-9 and abs(r["dy"]) < 1e-9 and r["chi2"] < 1e-15
    assert r["zm"] == pytest.approx(5287.6 + 0.0119379 * abs(xs) - 1418.42 * tx * tx, rel=1e-12)
    # |dty| exactly 0.02 fails, just below passes
    r = oracle64.match_pair([xs, ys - 0.02 * (10000 - 7826), tx, ty + 0.02], [1.0, 2.0, tx, ty])
    assert r["dty"] == pytest.approx(0.02) and r["presel"] == (1.0 if r["dty"] < 0.02 else 0.0)
    r = oracle64.match_pair([xs, ys, tx, ty + 0.0199], [1.0, 2.0, tx, ty])
    assert r["presel"] == 1.0
    r = oracle64.match_pair([xs + 20.5, ys, tx, ty], [1.0, 2.0, tx, ty])
    assert r["presel"] == 0.0
