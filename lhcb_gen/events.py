"""Seeded synthetic LHCb-like events (SciFi hits, VELO states, UT hits, truth).

Stands in for the paper's simulated samples, which are not
available.  One recipe serves the five BASELINE.json configs; DESIGN.md "Input
recipe" states it.  This module is shared by the oracle tests and the CUDA
tests; it holds the *toy track model used to make inputs* and none of the
reconstruction arithmetic.

Toy track model:
  * straight line from the vertex to the magnet, VELO state at z_velo;
  * one kick  dtx = polarity*q*K_B/p  at z_match of PAPER.md Eq. 18 (Table 1);
  * inside the SciFi  x(z) = ax + bx*zb + cx*zb^2*(1 + d_ratio*zb)  (Eq. 1) with
    cx = polarity*q*kappa/p, tangent to the post-kick line at z_scifi_state;
  * y is a straight line (L211, L231);
  * VELO->UT: x(z) = x + tx*dz + gamma*dz^2, gamma = A_g + B_g*polarity*q/p (Eq. 19-20).

Layout produced (all SoA, float32 unless noted):
  zone_off  u32[n_events*24+1]   zone index = (event*2 + half)*12 + layer, half 0: y > 0
  hit_x     f32[n_hits]          ascending inside each zone; stereo layers: x at y = 0
  hit_x64   f64[n_hits]          the same values before rounding (for f64 oracle checks)
  hit_pid   i32[n_hits]          global particle id, -1 for noise
  velo_off  u32[n_events+1];  velo_x, velo_y, velo_tx, velo_ty at z_velo;  velo_pid
  ut_off    u32[n_events*4+1];  ut_x0 ascending per (event, layer);  ut_ylo, ut_yhi;  ut_row u8;  ut_pid
  polarity  i8[n_events]
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Dict, Optional

import numpy as np

from .geometry import default_geom

N_LAYERS = 12
N_UT = 4
CHUNK = 1024

# Toy detector extents (BASELINE.json configs[1]; DESIGN.md input recipe)
SCIFI_X_MAX = 3000.0
SCIFI_Y_MAX = 2500.0
UT_X_MAX = 850.0
UT_Y_MAX = 700.0
UT_ROW = 100.0
UT_PITCH = 0.190
UT_STRIP0 = 4474                # strip number of x0 = 0


@dataclass
class GenConfig:
    name: str
    n_events: int
    seed: int
    tracks_mean: float = 200.0
    tracks_fixed: Optional[int] = None
    frac_long: float = 0.6          # of non-displaced tracks: VELO + UT + SciFi
    frac_displaced: float = 0.0
    noise_mean: float = 1500.0
    hit_eff: float = 0.98
    sigma_x: float = 0.080
    p_lo: float = 2000.0
    p_hi: float = 100000.0
    pt_min: float = 0.0
    slope_max: float = 0.25
    origin_sigma: float = 0.1
    ut: bool = True
    ut_noise: int = 3000
    polarity: str = "alternate"     # "down" | "up" | "alternate"
    # cfg5 only
    direct_seeds: bool = False
    seeds_mean: float = 250.0
    velo_mean: float = 350.0
    partner_frac: float = 0.7
    ut_total_mean: float = 5000.0


def config(idx: int, n_events: Optional[int] = None) -> GenConfig:
    """BASELINE.json configs[idx-1] (idx = 1..5)."""
    if idx == 1:
        c = GenConfig("cfg1", 16, 0, tracks_fixed=40, frac_long=1.0, noise_mean=0.0,
                      hit_eff=1.0, ut=False, ut_noise=0, polarity="down")
    elif idx == 2:
        c = GenConfig("cfg2", 1000, 1)
    elif idx == 3:
        c = GenConfig("cfg3", 16384, 2)
    elif idx == 4:
        c = GenConfig("cfg4", 2000, 3, tracks_mean=300.0, noise_mean=2500.0,
                      frac_displaced=0.2, p_lo=1500.0, pt_min=200.0)
    elif idx == 5:
        c = GenConfig("cfg5", 1000, 4, direct_seeds=True)
    else:
        raise ValueError("config index must be 1..5")
    if n_events is not None:
        c = replace(c, n_events=int(n_events))
    return c


@dataclass
class Events:
    n_events: int
    geom: dict
    cfg: GenConfig
    zone_off: np.ndarray
    hit_x: np.ndarray
    hit_x64: np.ndarray
    hit_pid: np.ndarray
    polarity: np.ndarray
    velo_off: np.ndarray
    velo_x: np.ndarray
    velo_y: np.ndarray
    velo_tx: np.ndarray
    velo_ty: np.ndarray
    velo_pid: np.ndarray
    ut_off: np.ndarray
    ut_x0: np.ndarray
    ut_ylo: np.ndarray
    ut_yhi: np.ndarray
    ut_pid: np.ndarray
    particles: Dict[str, np.ndarray] = field(default_factory=dict)
    ut_row: Optional[np.ndarray] = None       # u8 strip row per UT hit: y_lo = ut_row_y0 + row * ut_row_pitch
    ut_strip: Optional[np.ndarray] = None     # u16 strip number per UT hit: x0 = ut_strip_x0 + strip * ut_strip_pitch
    # cfg5: seeds given directly as states at z_scifi_state
    seed_off: Optional[np.ndarray] = None
    seed_state: Optional[np.ndarray] = None   # [5, n_seeds] x, y, tx, ty, qop
    seed_pid: Optional[np.ndarray] = None

    @property
    def n_hits(self) -> int:
        return int(self.hit_x.shape[0])


# --------------------------------------------------------------------------- toy model
def _g(zb, d):
    return zb * zb * (1.0 + d * zb)


def _gp(zb, d):
    return 2.0 * zb + 3.0 * d * zb * zb


def _kink_state(geom, pol, q, p, xv, yv, zv, tx0, ty):
    """VELO-plane state, post-kick SciFi state and Eq. 1 parameters (float64 arrays)."""
    zV, zS, zref, d = geom["z_velo"], geom["z_scifi_state"], geom["z_ref"], geom["d_ratio"]
    A, B, C, D, E = geom["mag"]
    x_V = xv + tx0 * (zV - zv)
    y_V = yv + ty * (zV - zv)
    dtx = pol * q * geom["kick_pt"] / p
    tx_S = tx0 + dtx
    x_S = x_V + tx0 * (zS - zV)
    for _ in range(12):     # D = 0.012: contraction, converges to double precision
        z_m = A + B * np.abs(dtx) + C * dtx * dtx + D * np.abs(x_S) + E * tx0 * tx0
        x_S = x_V + (z_m - zV) * tx0 + (zS - z_m) * tx_S
    cx = pol * q * geom["kappa_cx"] / p
    zbS = zS - zref
    bx = tx_S - cx * _gp(zbS, d)
    ax = x_S - bx * zbS - cx * _g(zbS, d)
    y_S = yv + ty * (zS - zv)
    return x_V, y_V, x_S, y_S, tx_S, ax, bx, cx


def _polarity(cfg: GenConfig, event_ids: np.ndarray) -> np.ndarray:
    if cfg.polarity == "down":
        return np.full(event_ids.shape, -1, np.int8)
    if cfg.polarity == "up":
        return np.full(event_ids.shape, +1, np.int8)
    return np.where(event_ids % 2 == 0, 1, -1).astype(np.int8)


def _sample_tracks(cfg: GenConfig, rng, n):
    q = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    p = np.exp(rng.uniform(np.log(cfg.p_lo), np.log(cfg.p_hi), n))
    tx0 = rng.uniform(-cfg.slope_max, cfg.slope_max, n)
    ty = rng.uniform(-cfg.slope_max, cfg.slope_max, n)
    return q, p, tx0, ty


def _ut_hits(geom, cfg, rng, pol_t, q, p, x_V, y_V, tx0, ty, zv, allowed, ev, pid):
    """True UT hits of the given tracks (Eq. 19-20), quantised to the strip pitch."""
    zV = geom["z_velo"]
    Ag, Bg = geom["gamma_ab"]
    gam = Ag + Bg * pol_t * q / p
    ev_l, lay_l, x0_l, ylo_l, yhi_l, pid_l = [], [], [], [], [], []
    for i in range(N_UT):
        dz = geom["ut_z"][i] - zV
        x = x_V + tx0 * dz + gam * dz * dz
        y = y_V + ty * dz
        ok = allowed & (zv < geom["ut_z"][i]) & (np.abs(x) < UT_X_MAX) & (np.abs(y) < UT_Y_MAX)
        ok &= rng.random(x.shape[0]) < cfg.hit_eff
        x0 = x - y * geom["ut_tan_alpha"][i]
        x0 = np.round(x0 / UT_PITCH) * UT_PITCH
        row = np.floor((y + UT_Y_MAX) / UT_ROW)
        ylo = -UT_Y_MAX + UT_ROW * row
        ev_l.append(ev[ok]); lay_l.append(np.full(int(ok.sum()), i, np.int64))
        x0_l.append(x0[ok]); ylo_l.append(ylo[ok]); yhi_l.append(ylo[ok] + UT_ROW)
        pid_l.append(pid[ok])
    return (np.concatenate(ev_l), np.concatenate(lay_l), np.concatenate(x0_l),
            np.concatenate(ylo_l), np.concatenate(yhi_l), np.concatenate(pid_l))


def _ut_noise(rng, ev):
    n = ev.shape[0]
    lay = rng.integers(0, N_UT, n)
    x0 = np.round(rng.uniform(-UT_X_MAX, UT_X_MAX, n) / UT_PITCH) * UT_PITCH
    row = rng.integers(0, int(2 * UT_Y_MAX / UT_ROW), n)
    ylo = -UT_Y_MAX + UT_ROW * row
    return ev, lay, x0, ylo, ylo + UT_ROW, np.full(n, -1, np.int64)


def _pack_ut(n_events, parts):
    ev = np.concatenate([p[0] for p in parts]); lay = np.concatenate([p[1] for p in parts])
    x0 = np.concatenate([p[2] for p in parts]); ylo = np.concatenate([p[3] for p in parts])
    yhi = np.concatenate([p[4] for p in parts]); pid = np.concatenate([p[5] for p in parts])
    zone = ev * N_UT + lay
    # strip numbers: the float x0 is DERIVED from them with the float32 operations the ABI states
    # (x0 = ut_strip_x0 + strip * ut_strip_pitch), so both forms of a UT hit agree bit for bit
    strip = (np.rint(x0 / UT_PITCH).astype(np.int64) + UT_STRIP0).astype(np.uint16)
    x0 = np.float32(-UT_STRIP0 * UT_PITCH) + strip.astype(np.float32) * np.float32(UT_PITCH)
    order = np.lexsort((strip, zone))
    off = np.zeros(n_events * N_UT + 1, np.uint32)
    np.cumsum(np.bincount(zone, minlength=n_events * N_UT), out=off[1:])
    # strip rows: one byte per hit.  The float form of the y coverage is DERIVED from the rows with the float32
    # operations the ABI states (y_lo = y0 + row * pitch, y_hi = y_lo + pitch), so both forms agree bit for bit.
    row = np.rint((ylo[order] + UT_Y_MAX) / UT_ROW).astype(np.uint8)
    ylo32 = np.float32(-UT_Y_MAX) + row.astype(np.float32) * np.float32(UT_ROW)
    yhi32 = ylo32 + np.float32(UT_ROW)
    return (off, x0[order].astype(np.float32), ylo32.astype(np.float32),
            yhi32.astype(np.float32), pid[order].astype(np.int32), row, strip[order])


def _empty_ut(n_events):
    z = np.zeros(0, np.float32)
    return np.zeros(n_events * N_UT + 1, np.uint32), z, z.copy(), z.copy(), np.zeros(0, np.int32), np.zeros(0, np.uint8), np.zeros(0, np.uint16)


def _shuffle_within(rng, ev):
    """Permutation that groups by event with random order inside each event."""
    return np.lexsort((rng.random(ev.shape[0]), ev))


def _gen_chunk(cfg: GenConfig, geom: dict, rng, n_events: int, event0: int):
    """One chunk of full events (SciFi + VELO + UT).  Event ids are local (0..n_events)."""
    d, zref = geom["d_ratio"], geom["z_ref"]
    if cfg.tracks_fixed is not None:
        n_trk = np.full(n_events, cfg.tracks_fixed, np.int64)
    else:
        n_trk = rng.poisson(cfg.tracks_mean, n_events)
    ev = np.repeat(np.arange(n_events), n_trk)
    N = ev.shape[0]
    pol_e = _polarity(cfg, np.arange(n_events) + event0)
    pol_t = pol_e[ev].astype(np.float64)

    q, p, tx0, ty = _sample_tracks(cfg, rng, N)
    u_kind, u_long = rng.random(N), rng.random(N)
    kind = np.where(u_kind < cfg.frac_displaced, 2, np.where(u_long < cfg.frac_long, 0, 1))
    xv = rng.normal(0.0, cfg.origin_sigma, N)
    yv = rng.normal(0.0, cfg.origin_sigma, N)
    zv = np.zeros(N)
    # displaced: vertex on a parent line from the origin, daughter within +-0.03 of the parent
    disp = kind == 2
    zv_d = rng.uniform(0.0, 2500.0, N)
    dtx_d, dty_d = rng.uniform(-0.03, 0.03, N), rng.uniform(-0.03, 0.03, N)
    xv = np.where(disp, tx0 * zv_d, xv); yv = np.where(disp, ty * zv_d, yv)
    zv = np.where(disp, zv_d, zv)
    tx0 = np.where(disp, tx0 + dtx_d, tx0); ty = np.where(disp, ty + dty_d, ty)
    if cfg.pt_min > 0.0:
        s2 = tx0 * tx0 + ty * ty
        p_need = cfg.pt_min * np.sqrt(1.0 + s2) / np.sqrt(np.maximum(s2, 1e-12))
        p = np.minimum(np.maximum(p, p_need), cfg.p_hi)

    x_V, y_V, x_S, y_S, tx_S, ax, bx, cx = _kink_state(geom, pol_t, q, p, xv, yv, zv, tx0, ty)

    # ---- SciFi hits -------------------------------------------------------
    z = np.asarray(geom["scifi_z"], np.float64)
    ta = np.asarray(geom["scifi_tan_alpha"], np.float64)
    zb = z - zref
    xt = ax[:, None] + bx[:, None] * zb[None, :] + cx[:, None] * _g(zb, d)[None, :]
    yt = yv[:, None] + ty[:, None] * (z[None, :] - zv[:, None])
    in_acc = (np.abs(xt) < SCIFI_X_MAX) & (np.abs(yt) < SCIFI_Y_MAX)
    rec = in_acc & (rng.random((N, N_LAYERS)) < cfg.hit_eff)
    meas = xt - yt * ta[None, :] + rng.normal(0.0, 1.0, (N, N_LAYERS)) * cfg.sigma_x
    half = np.where(yt > 0.0, 0, 1)
    ti, li = np.nonzero(rec)
    h_ev, h_half, h_lay = ev[ti], half[ti, li], li
    h_x, h_pid = meas[ti, li], ti

    n_noise = rng.poisson(cfg.noise_mean, n_events) if cfg.noise_mean > 0 else np.zeros(n_events, np.int64)
    nz_ev = np.repeat(np.arange(n_events), n_noise)
    M = nz_ev.shape[0]
    nz_lay = rng.integers(0, N_LAYERS, M)
    nz_x = rng.uniform(-SCIFI_X_MAX, SCIFI_X_MAX, M)
    nz_half = np.where(rng.uniform(-SCIFI_Y_MAX, SCIFI_Y_MAX, M) > 0.0, 0, 1)

    a_ev = np.concatenate([h_ev, nz_ev]); a_half = np.concatenate([h_half, nz_half])
    a_lay = np.concatenate([h_lay, nz_lay]); a_x = np.concatenate([h_x, nz_x])
    a_pid = np.concatenate([h_pid, np.full(M, -1, np.int64)])
    zone = (a_ev * 2 + a_half) * N_LAYERS + a_lay
    order = np.lexsort((a_x, zone))
    zone_off = np.zeros(n_events * 2 * N_LAYERS + 1, np.uint32)
    np.cumsum(np.bincount(zone, minlength=n_events * 2 * N_LAYERS), out=zone_off[1:])
    hit_x64 = a_x[order]
    hit_pid = a_pid[order].astype(np.int32)

    # ---- VELO states (long tracks only) -------------------------------------
    is_long = kind == 0
    vi = np.nonzero(is_long)[0]
    vi = vi[_shuffle_within(rng, ev[vi])]
    nv = vi.shape[0]
    sig_t = np.hypot(5e-5, 2.0 / p[vi])
    velo_x = x_V[vi] + rng.normal(0.0, 0.02, nv)
    velo_y = y_V[vi] + rng.normal(0.0, 0.02, nv)
    velo_tx = tx0[vi] + rng.normal(0.0, 1.0, nv) * sig_t
    velo_ty = ty[vi] + rng.normal(0.0, 1.0, nv) * sig_t
    velo_off = np.zeros(n_events + 1, np.uint32)
    np.cumsum(np.bincount(ev[vi], minlength=n_events), out=velo_off[1:])

    # ---- UT hits ---------------------------------------------------------------
    n_ut_true = np.zeros(N, np.int64)
    if cfg.ut:
        allowed = (kind == 0) | (kind == 2)
        true_ut = _ut_hits(geom, cfg, rng, pol_t, q, p, x_V, y_V, tx0, ty, zv, allowed,
                           ev, np.arange(N))
        np.add.at(n_ut_true, true_ut[5], 1)
        noise_ut = _ut_noise(rng, np.repeat(np.arange(n_events), cfg.ut_noise))
        ut = _pack_ut(n_events, [true_ut, noise_ut])
    else:
        ut = _empty_ut(n_events)

    # ---- truth table -------------------------------------------------------------
    is_x = ta == 0.0
    parts = dict(
        event=ev + event0, kind=kind.astype(np.int8), q=q.astype(np.int8), p=p,
        tx0=tx0, ty=ty, xv=xv, yv=yv, zv=zv, ax=ax, bx=bx, cx=cx,
        ay=yv + ty * (zref - zv), by=ty.copy(),
        x_S=x_S, y_S=y_S, tx_S=tx_S, x_V=x_V, y_V=y_V,
        n_x=rec[:, is_x].sum(1).astype(np.int8), n_uv=rec[:, ~is_x].sum(1).astype(np.int8),
        in_acc=in_acc.all(1),
        half_cross=(half.min(1) != half.max(1)),
        n_ut=n_ut_true.astype(np.int8),
        pol=pol_t.astype(np.int8),
    )
    return dict(
        n_events=n_events, n_particles=N, zone_off=zone_off, hit_x64=hit_x64, hit_pid=hit_pid,
        polarity=pol_e, velo_off=velo_off, velo_x=velo_x, velo_y=velo_y, velo_tx=velo_tx,
        velo_ty=velo_ty, velo_pid=vi.astype(np.int32), ut=ut, particles=parts,
    )


def _gen_chunk_direct(cfg: GenConfig, geom: dict, rng, n_events: int, event0: int):
    """cfg5: seeds given directly as SciFi states + VELO tracks + UT hits, no SciFi hits."""
    zS, zV, zy = geom["z_scifi_state"], geom["z_velo"], geom["z_match_y"]
    n_seed = rng.poisson(cfg.seeds_mean, n_events)
    n_velo = rng.poisson(cfg.velo_mean, n_events)
    ev = np.repeat(np.arange(n_events), n_seed)
    N = ev.shape[0]
    pol_e = _polarity(cfg, np.arange(n_events) + event0)
    pol_t = pol_e[ev].astype(np.float64)
    partner = rng.random(N) < cfg.partner_frac
    q, p, tx0, ty = _sample_tracks(cfg, rng, N)
    xv = rng.normal(0.0, cfg.origin_sigma, N); yv = rng.normal(0.0, cfg.origin_sigma, N)
    zv = np.zeros(N)
    x_V, y_V, x_S, y_S, tx_S, ax, bx, cx = _kink_state(geom, pol_t, q, p, xv, yv, zv, tx0, ty)
    # Gaussian residuals in the four matching variables, sized by the Eq. 23 tolerances
    f = geom["match_tol"]
    dtx = tx_S - tx0
    tol_x = f[0] * (f[1] ** 2 + f[2] ** 2 * dtx * dtx)
    tol_y = f[3] * (f[4] ** 2 + f[5] ** 2 * (tx0 * tx0 + ty * ty))
    r_x = rng.normal(0.0, 1.0, N) * 0.3 * np.sqrt(tol_x)
    r_y = rng.normal(0.0, 1.0, N) * 0.3 * np.sqrt(tol_y)
    r_ty = rng.normal(0.0, 1.0, N) * 0.3 * np.sqrt(1.0 / f[7])
    s_x = x_S + r_x
    s_tx = tx_S
    s_ty = ty + r_ty
    s_y = y_S + r_y - (zy - zS) * r_ty          # so that delta-y at z_match_y equals r_y
    s_qop = q / p
    # unpartnered seeds: random states
    rx = rng.uniform(-2500.0, 2500.0, N); ry = rng.uniform(-2000.0, 2000.0, N)
    rtx = rx / 5000.0 + rng.uniform(-0.3, 0.3, N); rty = ry / zS + rng.normal(0.0, 0.005, N)
    s_x = np.where(partner, s_x, rx); s_y = np.where(partner, s_y, ry)
    s_tx = np.where(partner, s_tx, rtx); s_ty = np.where(partner, s_ty, rty)
    seed_off = np.zeros(n_events + 1, np.uint32)
    np.cumsum(n_seed, out=seed_off[1:])
    seed_state = np.stack([s_x, s_y, s_tx, s_ty, s_qop]).astype(np.float32)
    seed_pid = np.where(partner, np.arange(N), -1).astype(np.int32)

    # VELO: partners' states plus random origin tracks up to Poisson(velo_mean)
    n_part = np.bincount(ev[partner], minlength=n_events)
    n_extra = np.maximum(n_velo - n_part, 0)
    e_ev = np.repeat(np.arange(n_events), n_extra)
    E = e_ev.shape[0]
    e_tx = rng.uniform(-cfg.slope_max, cfg.slope_max, E)
    e_ty = rng.uniform(-cfg.slope_max, cfg.slope_max, E)
    e_x = e_tx * zV + rng.normal(0.0, cfg.origin_sigma, E)
    e_y = e_ty * zV + rng.normal(0.0, cfg.origin_sigma, E)
    pi = np.nonzero(partner)[0]
    v_ev = np.concatenate([ev[pi], e_ev])
    v_x = np.concatenate([x_V[pi], e_x]); v_y = np.concatenate([y_V[pi], e_y])
    v_tx = np.concatenate([tx0[pi], e_tx]); v_ty = np.concatenate([ty[pi], e_ty])
    v_pid = np.concatenate([pi, np.full(E, -1, np.int64)])
    order = _shuffle_within(rng, v_ev)
    velo_off = np.zeros(n_events + 1, np.uint32)
    np.cumsum(np.bincount(v_ev, minlength=n_events), out=velo_off[1:])

    n_ut_true = np.zeros(N, np.int64)
    true_ut = _ut_hits(geom, cfg, rng, pol_t, q, p, x_V, y_V, tx0, ty, zv, partner, ev, np.arange(N))
    np.add.at(n_ut_true, true_ut[5], 1)
    n_tot = rng.poisson(cfg.ut_total_mean, n_events)
    n_noise = np.maximum(n_tot - np.bincount(true_ut[0], minlength=n_events), 0)
    noise_ut = _ut_noise(rng, np.repeat(np.arange(n_events), n_noise))
    ut = _pack_ut(n_events, [true_ut, noise_ut])

    parts = dict(event=ev + event0, kind=np.where(partner, 0, 1).astype(np.int8),
                 q=q.astype(np.int8), p=p, tx0=tx0, ty=ty, x_S=x_S, y_S=y_S, tx_S=tx_S,
                 x_V=x_V, y_V=y_V, n_ut=n_ut_true.astype(np.int8), pol=pol_t.astype(np.int8))
    return dict(
        n_events=n_events, n_particles=N,
        zone_off=np.zeros(n_events * 2 * N_LAYERS + 1, np.uint32),
        hit_x64=np.zeros(0), hit_pid=np.zeros(0, np.int32), polarity=pol_e,
        velo_off=velo_off, velo_x=v_x[order], velo_y=v_y[order], velo_tx=v_tx[order],
        velo_ty=v_ty[order], velo_pid=v_pid[order].astype(np.int32), ut=ut, particles=parts,
        seed_off=seed_off, seed_state=seed_state, seed_pid=seed_pid,
    )


def _cat_off(chunks, key, sub=None):
    """Concatenate prefix-offset arrays of consecutive chunks."""
    out, base = [np.zeros(1, np.uint64)], 0
    for c in chunks:
        o = (c[key] if sub is None else c[key][sub]).astype(np.uint64)
        out.append(o[1:] + base)
        base += int(o[-1])
    return np.concatenate(out).astype(np.uint32)


def _run_chunk(args):
    cfg, geom, k, e0, n = args
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([cfg.seed, k])))
    fn = _gen_chunk_direct if cfg.direct_seeds else _gen_chunk
    return fn(cfg, geom, rng, n, e0)


def generate(cfg: GenConfig, geom: Optional[dict] = None, workers: int = 1, first_chunk: int = 0) -> Events:
    """Generate cfg.n_events events, in independent chunks of CHUNK events.

    Chunk k draws from numpy's PCG64 seeded with SeedSequence([cfg.seed, k]), so a full chunk does
    not depend on how many chunks follow it (cfg3 batch slicing).  `first_chunk` shifts the chunk
    indices (rank r of a multi-GPU run takes its own chunk range).  `workers` > 1 generates chunks
    in parallel processes; the result is identical.
    """
    geom = default_geom() if geom is None else geom
    jobs = []
    for j, e0 in enumerate(range(0, cfg.n_events, CHUNK)):
        jobs.append((cfg, geom, first_chunk + j, first_chunk * CHUNK + e0, min(CHUNK, cfg.n_events - e0)))
    if workers > 1 and len(jobs) > 1:
        import multiprocessing as mp
        with mp.get_context("fork").Pool(min(workers, len(jobs))) as pool:
            chunks = pool.map(_run_chunk, jobs)
    else:
        chunks = [_run_chunk(j) for j in jobs]
    pid_base = 0
    for c in chunks:
        for key in ("hit_pid", "velo_pid", "seed_pid"):
            if key in c and c[key] is not None:
                c[key] = np.where(c[key] >= 0, c[key] + pid_base, -1).astype(np.int32)
        u = list(c["ut"]); u[4] = np.where(u[4] >= 0, u[4] + pid_base, -1).astype(np.int32)
        c["ut"] = tuple(u)
        pid_base += c["n_particles"]

    cat = lambda key: np.concatenate([c[key] for c in chunks])
    hit_x64 = cat("hit_x64")
    parts = {k: np.concatenate([c["particles"][k] for c in chunks]) for k in chunks[0]["particles"]}
    evs = Events(
        n_events=cfg.n_events, geom=geom, cfg=cfg,
        zone_off=_cat_off(chunks, "zone_off"),
        hit_x=hit_x64.astype(np.float32), hit_x64=hit_x64, hit_pid=cat("hit_pid"),
        polarity=cat("polarity"),
        velo_off=_cat_off(chunks, "velo_off"),
        velo_x=cat("velo_x").astype(np.float32), velo_y=cat("velo_y").astype(np.float32),
        velo_tx=cat("velo_tx").astype(np.float32), velo_ty=cat("velo_ty").astype(np.float32),
        velo_pid=cat("velo_pid"),
        ut_off=_cat_off(chunks, "ut", 0),
        ut_x0=np.concatenate([c["ut"][1] for c in chunks]),
        ut_ylo=np.concatenate([c["ut"][2] for c in chunks]),
        ut_yhi=np.concatenate([c["ut"][3] for c in chunks]),
        ut_pid=np.concatenate([c["ut"][4] for c in chunks]),
        particles=parts,
        ut_row=np.concatenate([c["ut"][5] for c in chunks]),
        ut_strip=np.concatenate([c["ut"][6] for c in chunks]),
    )
    if cfg.direct_seeds:
        evs.seed_off = _cat_off(chunks, "seed_off")
        evs.seed_state = np.concatenate([c["seed_state"] for c in chunks], axis=1)
        evs.seed_pid = cat("seed_pid")
    return evs


def slice_events(ev: Events, start: int, stop: int) -> Events:
    """Events [start, stop) as a self-contained Events (offsets rebased; pids unchanged)."""
    z0, z1 = start * 24, stop * 24
    h0, h1 = int(ev.zone_off[z0]), int(ev.zone_off[z1])
    v0, v1 = int(ev.velo_off[start]), int(ev.velo_off[stop])
    u0, u1 = int(ev.ut_off[start * 4]), int(ev.ut_off[stop * 4])
    out = replace(
        ev, n_events=stop - start,
        zone_off=(ev.zone_off[z0:z1 + 1] - ev.zone_off[z0]).astype(np.uint32),
        hit_x=ev.hit_x[h0:h1], hit_x64=ev.hit_x64[h0:h1], hit_pid=ev.hit_pid[h0:h1],
        polarity=ev.polarity[start:stop],
        velo_off=(ev.velo_off[start:stop + 1] - ev.velo_off[start]).astype(np.uint32),
        velo_x=ev.velo_x[v0:v1], velo_y=ev.velo_y[v0:v1], velo_tx=ev.velo_tx[v0:v1],
        velo_ty=ev.velo_ty[v0:v1], velo_pid=ev.velo_pid[v0:v1],
        ut_off=(ev.ut_off[start * 4:stop * 4 + 1] - ev.ut_off[start * 4]).astype(np.uint32),
        ut_x0=ev.ut_x0[u0:u1], ut_ylo=ev.ut_ylo[u0:u1], ut_yhi=ev.ut_yhi[u0:u1],
        ut_pid=ev.ut_pid[u0:u1], ut_row=ev.ut_row[u0:u1] if ev.ut_row is not None else None,
        ut_strip=ev.ut_strip[u0:u1] if ev.ut_strip is not None else None,
    )
    if ev.seed_off is not None:
        s0, s1 = int(ev.seed_off[start]), int(ev.seed_off[stop])
        out.seed_off = (ev.seed_off[start:stop + 1] - ev.seed_off[start]).astype(np.uint32)
        out.seed_state = ev.seed_state[:, s0:s1]
        out.seed_pid = ev.seed_pid[s0:s1]
    return out
