"""Pins of the ghost-killing network in the oracle (reading A14b)."""
import numpy as np
import pytest

from lhcb_gen import config, default_geom, generate, ghost_nn
from lhcb_gen.ghost_nn import unpack
from oracle.binding import Oracle


@pytest.fixture(scope="module")
def o32():
    return Oracle(default_geom(), "f32")


def test_spelled_out_exp_and_log_against_libm(o32):
    ys = np.linspace(-30, 30, 2001)
    e = np.array([o32.spec_exp(y) for y in ys])
    assert np.max(np.abs(e / np.exp(ys.astype(np.float32).astype(np.float64)) - 1)) < 6e-7      # measured 2.3e-7
    assert o32.spec_exp(0.0) == 1.0
    assert o32.spec_exp(-1000.0) == o32.spec_exp(-87.0) and o32.spec_exp(1000.0) == o32.spec_exp(87.0)   # clamped
    xs = np.exp(np.linspace(-12, 12, 2001)).astype(np.float32).astype(np.float64)
    l = np.array([o32.spec_log(x) for x in xs])
    assert np.max(np.abs(l - np.log(xs))) < 2e-6                                                # measured 1.0e-6
    assert o32.spec_log(1.0) == 0.0
    o64 = Oracle(default_geom(), "f64")
    assert abs(o64.spec_log(7.5) - np.log(7.5)) < 1e-7 and abs(o64.spec_exp(1.0) / np.e - 1) < 1e-6
    # in float64 what is left is the truncation of the two series: degree 6 on |r| <= ln2 / 2 (1.6e-7), five terms
    # of the atanh series on |s| <= 0.172 (3.3e-8); a wider reduction interval or a dropped term shows at once
    e64 = np.array([o64.spec_exp(y) for y in ys])
    assert np.max(np.abs(e64 / np.exp(ys) - 1)) < 2.5e-7
    l64 = np.array([o64.spec_log(x) for x in xs])
    assert np.max(np.abs(l64 - np.log(xs))) < 6e-8


def test_eta_is_the_pseudorapidity(o32):
    for tx, ty in [(0.1, 0.0), (0.0, -0.02), (0.25, 0.25), (0.003, 0.004), (-0.05, 0.12)]:
        theta = np.arctan(np.hypot(tx, ty))
        assert abs(o32.eta_velo(tx, ty) + np.log(np.tan(theta / 2))) < 5e-6 * (1 + abs(np.log(np.tan(theta / 2))))


def test_ghost_prob_is_the_mlp(o32):
    """8 -> 32 (ReLU) -> 1 (logistic) on standardised inputs, against a numpy float64 evaluation."""
    rng = np.random.default_rng(3)
    for trial in range(20):
        w = np.concatenate([rng.normal(0, 1, 8), rng.uniform(0.5, 2, 8), rng.normal(0, 0.5, 256), rng.normal(0, 0.5, 32),
                            rng.normal(0, 0.5, 32), rng.normal(0, 1, 1), [0.8, 0.05]]).astype(np.float32)
        x = rng.normal(0, 2, 8).astype(np.float32)
        n = unpack(w.astype(np.float64))
        u = (x.astype(np.float64) - n["mu"]) * n["isig"]
        t = n["b2"] + n["W2"] @ np.maximum(n["W1"] @ u + n["b1"], 0)
        assert abs(o32.ghost_prob(w, x) - 1 / (1 + np.exp(-t))) < 2e-5
    # special cases: all-zero weights -> 1/2 exactly; a dropped hidden bias or a transposed W1 would show above
    z = np.zeros(339, np.float32); z[8:16] = 1
    assert o32.ghost_prob(z, np.ones(8)) == 0.5
    z[336] = 3.0
    assert abs(o32.ghost_prob(z, np.ones(8)) - 1 / (1 + np.exp(-3.0))) < 1e-6


def run(o, ev, nn):
    s = o.seeding(ev)
    seed_off = np.zeros(ev.n_events + 1, np.uint32)
    np.cumsum(np.bincount(s["event"], minlength=ev.n_events), out=seed_off[1:])
    nhits = (s["nx"] + s["nuv"]).astype(np.uint8)
    return s, seed_off, nhits, o.matching(ev.n_events, seed_off, s["state"], ev, use_ut=True, nn=nn, nhits=nhits)


def test_selection_equals_the_literal_rule_of_L348():
    """Brute force in Python from the unfiltered candidate list: keep p < 0.8; drop a track that shares its
    seed or its VELO segment with another kept track whose ghost probability is lower by >= 0.05."""
    ev = generate(config(2, 40))
    o = Oracle(ev.geom, "f32")
    w = ghost_nn()
    open_w = w.copy(); open_w[337] = np.inf; open_w[338] = np.inf
    s, seed_off, nhits, allc = run(o, ev, open_w)
    _, _, _, sel = run(o, ev, w)
    # every candidate's ghost probability = the MLP on its own features
    for i in range(0, allc["n"], 97):
        sd, v = allc["seed"][i], allc["velo"][i]
        r = o.match_pair(s["state"][sd, :4], [ev.velo_x[v], ev.velo_y[v], ev.velo_tx[v], ev.velo_ty[v]])
        x = [r["zm"], r["dx"], r["dy"], r["dtx"], r["dty"], r["chi2"], o.eta_velo(ev.velo_tx[v], ev.velo_ty[v]), nhits[sd]]
        assert abs(o.ghost_prob(w, x) - allc["ghost"][i]) < 1e-6
    cut, margin = np.float32(w[337]), np.float32(w[338])
    p = allc["ghost"].astype(np.float32)
    kept = p < cut
    expect = set()
    for i in np.flatnonzero(kept):
        share = kept & ((allc["seed"] == allc["seed"][i]) | (allc["velo"] == allc["velo"][i]))
        share[i] = False
        if not (p[i] >= (p[share] + margin).astype(np.float32)).any():
            expect.add((int(allc["seed"][i]), int(allc["velo"][i])))
    got = set(zip(sel["seed"].tolist(), sel["velo"].tolist()))
    assert got == expect and len(got) > 50 * 40
    assert (sel["ghost"] < cut).all()
    assert len(got) < allc["n"]                                 # the selection does remove something
    # a flat network (outputs squeezed around 1/2, all below the cut) with a 0.004 margin: now the margin decides
    # some twenty removals (few seeds have two candidates), so a misread margin or comparison set shows
    flat = w.copy(); flat[304:336] *= 0.02; flat[336] = 0.0; flat[337] = 0.8; flat[338] = 0.004
    open_f = flat.copy(); open_f[337] = np.inf; open_f[338] = np.inf
    _, _, _, allf = run(o, ev, open_f)
    _, _, _, self_ = run(o, ev, flat)
    pf = allf["ghost"].astype(np.float32)
    assert (pf < 0.8).all() and pf.std() > 0.002
    expect_f, removed_by_margin = set(), 0
    for i in range(allf["n"]):
        share = (allf["seed"] == allf["seed"][i]) | (allf["velo"] == allf["velo"][i])
        share[i] = False
        if (pf[i] >= (pf[share] + np.float32(0.004)).astype(np.float32)).any():
            removed_by_margin += 1
        else:
            expect_f.add((int(allf["seed"][i]), int(allf["velo"][i])))
    assert set(zip(self_["seed"].tolist(), self_["velo"].tolist())) == expect_f and removed_by_margin >= 10
    # without the network the chi2 ranking (A14) is unchanged
    m0 = o.matching(ev.n_events, seed_off, s["state"], ev, use_ut=True)
    assert "ghost" not in m0 and m0["n"] > 0


def literal_selection(allc, cut, margin):
    """PAPER.md L348 word for word, in float32: kept if "smaller than" the cut; removed if another kept track with
    the same seed or the same VELO segment has a ghost probability "at least" `margin` lower."""
    p = allc["ghost"].astype(np.float32)
    kept = p < np.float32(cut)
    out = set()
    for i in np.flatnonzero(kept):
        share = kept & ((allc["seed"] == allc["seed"][i]) | (allc["velo"] == allc["velo"][i]))
        share[i] = False
        if not (p[i] >= (p[share] + np.float32(margin)).astype(np.float32)).any():
            out.add((int(allc["seed"][i]), int(allc["velo"][i])))
    return out


def exact_edge_cases(allc):
    """From the unfiltered candidates: (i, cut) with cut = candidate i's own probability, and (i, j, margin) with
    i and j sharing a segment, p_j < p_i <= 2 p_j (so that p_i - p_j and p_j + (p_i - p_j) are exact in float32:
    the sum lands exactly on p_i), every other competitor of i being too high to matter."""
    p = allc["ghost"].astype(np.float32)
    i_cut = int(np.argsort(p)[len(p) // 2])
    for i in range(allc["n"]):
        share = (allc["seed"] == allc["seed"][i]) | (allc["velo"] == allc["velo"][i])
        share[i] = False
        js = np.flatnonzero(share)
        if len(js) == 0:
            continue
        j = int(js[np.argmin(p[js])])
        if not (p[j] < p[i] <= 2 * p[j]):
            continue
        m = np.float32(p[i] - p[j])
        others = js[js != j]
        if np.float32(p[j] + m) == p[i] and (np.float32(1) * (p[others] + m) > p[i]).all():
            return i_cut, p[i_cut], i, j, m
    raise AssertionError("no pair of candidates for the margin edge")


def test_cut_is_strict_and_margin_is_inclusive_on_exact_float32_edges():
    """ghost probability "smaller than 0.8" (a track AT the cut is dropped) and "at least 0.05
    higher" (a track EXACTLY the margin above its competitor is removed).  Cut and margin are inputs, so both
    edges can be hit exactly: the cut is set to a candidate's own probability, the margin to the float32
    difference of two candidates that share a segment."""
    ev = generate(config(2, 12))
    o = Oracle(ev.geom, "f32")
    # the flat network of the test above: probabilities squeezed around 1/2, so that tracks sharing a segment are
    # within a factor two of each other
    w = ghost_nn(); w[304:336] *= 0.02; w[336] = 0.0
    open_w = w.copy(); open_w[337] = np.inf; open_w[338] = np.inf
    _, _, _, allc = run(o, ev, open_w)
    i_cut, p_cut, i, j, m = exact_edge_cases(allc)
    key = lambda k: (int(allc["seed"][k]), int(allc["velo"][k]))
    sel_of = lambda r: set(zip(r["seed"].tolist(), r["velo"].tolist()))
    # the cut: at the candidate's own probability it is dropped, one float32 step above it is kept
    for cut, kept in ((p_cut, False), (np.nextafter(p_cut, np.float32(2)), True)):
        nn = w.copy(); nn[337] = cut; nn[338] = np.inf
        got = sel_of(run(o, ev, nn)[3])
        assert (key(i_cut) in got) == kept, (cut, kept)
        assert got == literal_selection(allc, cut, np.inf)
    # the margin: exactly p_i - p_j removes i, the next margin that lifts the sum past p_i keeps it (no other competitor of
    # i is that low)
    pi, pj = np.float32(allc["ghost"][i]), np.float32(allc["ghost"][j])
    m_above = np.float32(np.nextafter(pi, np.float32(2)) - pj)        # the smallest margin whose float32 sum with p_j exceeds p_i
    for margin, kept in ((m, False), (m_above, True)):
        assert (np.float32(pj + np.float32(margin)) > pi) == kept
        nn = w.copy(); nn[337] = np.inf; nn[338] = margin
        got = sel_of(run(o, ev, nn)[3])
        assert (key(i) in got) == kept and key(j) in got, (margin, kept)
        assert got == literal_selection(allc, np.inf, margin)
