"""ctypes binding of the CPU oracle (TEST INFRASTRUCTURE).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

NO_HIT = 0xFFFFFFFF
COUNTER_NAMES = ["t1_hits", "pairs", "triplets", "ext_ok", "fit_ok", "xz_kept", "uv_first", "uv_steps",
                 "y_fits", "seeds", "sv_pairs", "presel", "chi2_ok", "ut_steps", "ut_hyp", "long"]

D, I = C.c_double, C.c_int32


class OrcGeom(C.Structure):
    _fields_ = [
        ("scifi_z", D * 12), ("scifi_tan_alpha", D * 12), ("z_ref", D), ("d_ratio", D),
        ("p_min", D), ("inv_p_a", D), ("inv_p_b", D), ("alpha0", D), ("alpha1", D),
        ("iter_layers", (I * 3) * 2), ("kappa_cx", D), ("cx_band", D * 4),
        ("tol_x_ext", D), ("tol_uv", D), ("min_x_hits", I), ("min_uv_hits", I),
        ("uv_first_layer", I * 2), ("sigma_hit", D), ("chi2x_max", D), ("chi2y_max", D),
        ("y_min", D), ("y_max", D), ("y_half_tol", D),
        ("z_velo", D), ("z_scifi_state", D), ("z_match_y", D),
        ("mag", D * 5), ("gamma_ab", D * 2), ("kick_pt", D), ("polarity", I),
        ("presel", D * 4), ("match_tol", D * 8), ("chi2_match_max", D),
        ("ut_z", D * 4), ("ut_tan_alpha", D * 4), ("ut_loose", (D * 4) * 4), ("ut_tight", (D * 4) * 4),
        ("ut_y_tol", D), ("min_ut_hits", I), ("ut_enabled", I),
    ]


def _fill(struct, geom: dict):
    for name, ctype in struct._fields_:
        v = geom[name]
        if isinstance(v, (list, tuple)):
            arr = getattr(struct, name)
            for i, vi in enumerate(v):
                if isinstance(vi, (list, tuple)):
                    for j, vj in enumerate(vi):
                        arr[i][j] = vj
                else:
                    arr[i] = vi
        else:
            setattr(struct, name, v)
    return struct


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


class Oracle:
    """mode: 'f32' (spec mode, decides parity) or 'f64' (truth recovery)."""

    def __init__(self, geom: dict, mode: str = "f32"):
        _build.build()
        self.mode = mode
        self.real = np.float32 if mode == "f32" else np.float64
        self.creal = C.c_float if mode == "f32" else C.c_double
        self.lib = C.CDLL(_build.lib_path(mode))
        L = self.lib
        L.orc_ctx_size.restype = C.c_size_t
        L.orc_seeding.restype = C.c_int64
        L.orc_matching.restype = C.c_int64
        L.orc_matching_nn.restype = C.c_int64
        for fn in (L.orc_spec_exp, L.orc_spec_log):
            fn.restype = D; fn.argtypes = [D]
        L.orc_eta_velo.restype = D; L.orc_eta_velo.argtypes = [D, D]
        L.orc_ghost_prob.restype = D
        L.orc_ghost_prob.argtypes = [C.POINTER(D), C.POINTER(D)]
        L.orc_clone_key.restype = C.c_uint64
        L.orc_clone_key.argtypes = [D, D, C.c_int, C.c_int]
        L.orc_ut_window.restype = D
        L.orc_ut_window.argtypes = [C.c_void_p, C.c_int, C.c_int, D]
        L.orc_gamma.restype = D
        L.orc_gamma.argtypes = [C.c_void_p, D]
        assert L.orc_real_size() == np.dtype(self.real).itemsize
        self.geom = geom
        self._g = _fill(OrcGeom(), geom)
        self._ctx = C.create_string_buffer(L.orc_ctx_size())
        rc = L.orc_init(C.byref(self._g), self._ctx)
        if rc != 0:
            raise ValueError(f"orc_init failed: {rc}")
        self.ctx = C.cast(self._ctx, C.c_void_p)

    # ------------------------------------------------------------------ batch calls
    def _hits(self, ev):
        return np.ascontiguousarray(ev.hit_x if self.mode == "f32" else ev.hit_x64, dtype=self.real)

    def seeding(self, ev, cap: int | None = None):
        hx = self._hits(ev)
        cap = cap or max(1024, 600 * ev.n_events)
        o_event = np.zeros(cap, np.int32); o_half = np.zeros(cap, np.int32)
        o_state = np.zeros((cap, 5), self.real); o_par = np.zeros((cap, 7), self.real)
        o_hits = np.zeros((cap, 12), np.uint32); o_nx = np.zeros(cap, np.uint8); o_nuv = np.zeros(cap, np.uint8)
        cnt = np.zeros(len(COUNTER_NAMES), np.uint64)
        zo = np.ascontiguousarray(ev.zone_off, np.uint32)
        pol = np.ascontiguousarray(ev.polarity, np.int8)
        n = self.lib.orc_seeding(self.ctx, C.c_int(ev.n_events), _p(zo, C.c_uint32), _p(hx, self.creal),
                                 _p(pol, C.c_int8), C.c_int64(cap), _p(o_event, C.c_int32), _p(o_half, C.c_int32),
                                 _p(o_state, self.creal), _p(o_par, self.creal), _p(o_hits, C.c_uint32),
                                 _p(o_nx, C.c_uint8), _p(o_nuv, C.c_uint8), _p(cnt, C.c_uint64))
        if n > cap:
            raise RuntimeError(f"oracle seed capacity {cap} < {n}")
        return dict(n=n, event=o_event[:n], half=o_half[:n], state=o_state[:n], par=o_par[:n], hits=o_hits[:n],
                    nx=o_nx[:n], nuv=o_nuv[:n], counters=dict(zip(COUNTER_NAMES, cnt.tolist())))

    def matching(self, n_events, seed_off, state, ev, use_ut=True, cap: int | None = None, nn=None, nhits=None,
                 hits=None):
        """seed_off u32[n_events+1], state [n][5]; VELO/UT/polarity from ev.
        hits: u32 [n][12] hit indices of the seeds (exact chi2 ties between twin seeds are then broken by the
        hit lists, reading A21) or None (ties to the lower seed index).
        nn: the 339 packed values of the ghost-killing network (reading A14b) or None (A14: chi2 ranking);
        nhits: u8 per seed (nHits_SciFi), None = 12."""
        cap = cap or max(1024, 400 * n_events)
        r = self.real
        state = np.ascontiguousarray(state, r)
        so = np.ascontiguousarray(seed_off, np.uint32)
        vo = np.ascontiguousarray(ev.velo_off, np.uint32)
        vx, vy, vtx, vty = (np.ascontiguousarray(a, r) for a in (ev.velo_x, ev.velo_y, ev.velo_tx, ev.velo_ty))
        if use_ut and len(ev.ut_x0):
            uo = np.ascontiguousarray(ev.ut_off, np.uint32)
            ux, ul, uh = (np.ascontiguousarray(a, r) for a in (ev.ut_x0, ev.ut_ylo, ev.ut_yhi))
        else:
            uo = ux = ul = uh = None
        pol = np.ascontiguousarray(ev.polarity, np.int8)
        o_event = np.zeros(cap, np.int32); o_seed = np.zeros(cap, np.uint32); o_velo = np.zeros(cap, np.uint32)
        o_ut = np.zeros((cap, 4), np.uint32); o_nut = np.zeros(cap, np.uint8)
        o_qop = np.zeros(cap, r); o_chi2 = np.zeros(cap, r)
        cnt = np.zeros(len(COUNTER_NAMES), np.uint64)
        if nn is not None:
            nnr = np.ascontiguousarray(nn, r)
            assert nnr.size == 339
            nh = np.ascontiguousarray(nhits, np.uint8) if nhits is not None else None
            o_ghost = np.zeros(cap, r)
            n = self.lib.orc_matching_nn(self.ctx, C.c_int(n_events), _p(so, C.c_uint32), _p(state, self.creal),
                                         _p(vo, C.c_uint32), _p(vx, self.creal), _p(vy, self.creal), _p(vtx, self.creal),
                                         _p(vty, self.creal), _p(uo, C.c_uint32), _p(ux, self.creal), _p(ul, self.creal),
                                         _p(uh, self.creal), _p(pol, C.c_int8), C.c_int64(cap), _p(o_event, C.c_int32),
                                         _p(o_seed, C.c_uint32), _p(o_velo, C.c_uint32), _p(o_ut, C.c_uint32),
                                         _p(o_nut, C.c_uint8), _p(o_qop, self.creal), _p(o_chi2, self.creal),
                                         _p(cnt, C.c_uint64), _p(nh, C.c_uint8), _p(nnr, self.creal), _p(o_ghost, self.creal))
            if n > cap:
                raise RuntimeError(f"oracle long-track capacity {cap} < {n}")
            return dict(n=n, event=o_event[:n], seed=o_seed[:n], velo=o_velo[:n], ut=o_ut[:n], n_ut=o_nut[:n],
                        qop=o_qop[:n], chi2=o_chi2[:n], ghost=o_ghost[:n],
                        counters=dict(zip(COUNTER_NAMES, cnt.tolist())))
        n = self.lib.orc_matching(self.ctx, C.c_int(n_events), _p(so, C.c_uint32), _p(state, self.creal),
                                  _p(vo, C.c_uint32), _p(vx, self.creal), _p(vy, self.creal), _p(vtx, self.creal),
                                  _p(vty, self.creal), _p(uo, C.c_uint32), _p(ux, self.creal), _p(ul, self.creal),
                                  _p(uh, self.creal), _p(pol, C.c_int8), C.c_int64(cap), _p(o_event, C.c_int32),
                                  _p(o_seed, C.c_uint32), _p(o_velo, C.c_uint32), _p(o_ut, C.c_uint32),
                                  _p(o_nut, C.c_uint8), _p(o_qop, self.creal), _p(o_chi2, self.creal),
                                  _p(cnt, C.c_uint64),
                                  _p(np.ascontiguousarray(hits, np.uint32), C.c_uint32) if hits is not None else None)
        if n > cap:
            raise RuntimeError(f"oracle long-track capacity {cap} < {n}")
        return dict(n=n, event=o_event[:n], seed=o_seed[:n], velo=o_velo[:n], ut=o_ut[:n], n_ut=o_nut[:n],
                    qop=o_qop[:n], chi2=o_chi2[:n], counters=dict(zip(COUNTER_NAMES, cnt.tolist())))

    def reconstruct(self, ev, use_ut=True):
        """Seeding followed by matching on the oracle's own seeds."""
        s = self.seeding(ev)
        seed_off = np.zeros(ev.n_events + 1, np.uint32)
        np.cumsum(np.bincount(s["event"], minlength=ev.n_events), out=seed_off[1:])
        m = self.matching(ev.n_events, seed_off, s["state"], ev, use_ut=use_ut, hits=s["hits"])
        return s, m

    def set_uv_hough(self, on: bool):
        """Hough-cluster UV seeding (reading A20) instead of the iterative default."""
        self.lib.orc_set_uv_hough(self.ctx, C.c_int(1 if on else 0))

    def hough_constants(self):
        o = self._dout(4); self.lib.orc_hough_constants(self.ctx, _p(o, D))
        return dict(zip(["tlo0", "tlo1", "w", "invw"], o))

    # ------------------------------------------------------------------ probes (pins)
    def spec_exp(self, y): return self.lib.orc_spec_exp(float(y))
    def spec_log(self, x): return self.lib.orc_spec_log(float(x))
    def eta_velo(self, tx, ty): return self.lib.orc_eta_velo(float(tx), float(ty))

    def ghost_prob(self, nn, inputs):
        a = np.ascontiguousarray(nn, np.float64); b = np.ascontiguousarray(inputs, np.float64)
        assert a.size == 339 and b.size == 8
        return self.lib.orc_ghost_prob(_p(a, D), _p(b, D))

    def seeding_debug(self, ev, event, half, cap_t=200000, cap_c=50000):
        hx = self._hits(ev)
        zo = np.ascontiguousarray(ev.zone_off, np.uint32)
        nt, nc = C.c_int64(0), C.c_int64(0)
        t_it = np.zeros(cap_t, np.int32); t_idx = np.zeros((cap_t, 3), np.uint32)
        c_par = np.zeros((cap_c, 4), self.real); c_hits = np.zeros((cap_c, 6), np.uint32)
        c_nx = np.zeros(cap_c, np.int32); c_it = np.zeros(cap_c, np.int32)
        c_key = np.zeros(cap_c, np.uint64); c_keep = np.zeros(cap_c, np.int32)
        self.lib.orc_seeding_debug(self.ctx, _p(zo, C.c_uint32), _p(hx, self.creal), C.c_int(event), C.c_int(half),
                                   C.c_int64(cap_t), C.byref(nt), _p(t_it, C.c_int32), _p(t_idx, C.c_uint32),
                                   C.c_int64(cap_c), C.byref(nc), _p(c_par, self.creal), _p(c_hits, C.c_uint32),
                                   _p(c_nx, C.c_int32), _p(c_it, C.c_int32), _p(c_key, C.c_uint64),
                                   _p(c_keep, C.c_int32))
        nt, nc = nt.value, nc.value
        assert nt <= cap_t and nc <= cap_c
        return dict(t_it=t_it[:nt], t_idx=t_idx[:nt], c_par=c_par[:nc], c_hits=c_hits[:nc], c_nx=c_nx[:nc],
                    c_it=c_it[:nc], c_key=c_key[:nc], c_keep=c_keep[:nc])

    def _dout(self, n):
        return np.zeros(n, np.float64)

    def constants(self):
        o = self._dout(16); self.lib.orc_constants(self.ctx, _p(o, D))
        return dict(dx3max=o[0:2], alpha_corr=o[2:4], K=o[4:6], r13=o[6:8])

    def pinv_xz(self, pattern):
        o = self._dout(18); self.lib.orc_pinv_xz(self.ctx, C.c_int(pattern), _p(o, D)); return o.reshape(3, 6)

    def pinv_y(self, mask):
        o = self._dout(12); self.lib.orc_pinv_y(self.ctx, C.c_int(mask), _p(o, D)); return o.reshape(2, 6)

    def momentum(self, it, x1, x3):
        o = self._dout(7); self.lib.orc_momentum(self.ctx, C.c_int(it), D(x1), D(x3), _p(o, D))
        return dict(zip(["t13", "x0", "s", "invp", "x2c", "lo2", "hi2"], o))

    def parabola3(self, it, x1, x2, x3):
        o = self._dout(3); self.lib.orc_parabola3(self.ctx, C.c_int(it), D(x1), D(x2), D(x3), _p(o, D)); return o

    def fit_xz(self, it, xs, missing_slot=-1):
        xs = np.ascontiguousarray(xs, np.float64); o = self._dout(4)
        self.lib.orc_fit_xz(self.ctx, C.c_int(it), _p(xs, D), C.c_int(missing_slot), _p(o, D)); return o

    def fit_y(self, mask, m):
        m = np.ascontiguousarray(m, np.float64); o = self._dout(3)
        self.lib.orc_fit_y(self.ctx, C.c_int(mask), _p(m, D), _p(o, D)); return o

    def clone_key(self, chi2, cx, nx, it=0):
        return int(self.lib.orc_clone_key(D(chi2), D(cx), C.c_int(nx), C.c_int(it)))

    def clone_kill(self, keys, hits, nx, nhits):
        keys = np.ascontiguousarray(keys, np.uint64); hits = np.ascontiguousarray(hits, np.uint32)
        nx = np.ascontiguousarray(nx, np.int32); keep = np.zeros(len(keys), np.int32)
        self.lib.orc_clone_kill(C.c_int(len(keys)), _p(keys, C.c_uint64), _p(hits, C.c_uint32), _p(nx, C.c_int32),
                                C.c_uint32(nhits), _p(keep, C.c_int32))
        return keep.astype(bool)

    def match_pair(self, seed4, velo4):
        s = np.ascontiguousarray(seed4, np.float64); v = np.ascontiguousarray(velo4, np.float64); o = self._dout(7)
        self.lib.orc_match_pair(self.ctx, _p(s, D), _p(v, D), _p(o, D))
        return dict(zip(["dx", "dy", "dtx", "dty", "zm", "chi2", "presel"], o))

    def ut_window(self, layer, tight, invp_gev):
        return float(self.lib.orc_ut_window(self.ctx, C.c_int(layer), C.c_int(int(tight)), D(invp_gev)))

    def gamma(self, q0):
        return float(self.lib.orc_gamma(self.ctx, D(q0)))

    def ut_search(self, velo4, q0, ut_off5, ux, uylo, uyhi):
        v = np.ascontiguousarray(velo4, np.float64)
        uo = np.ascontiguousarray(ut_off5, np.uint32)
        ux, ul, uh = (np.ascontiguousarray(a, self.real) for a in (ux, uylo, uyhi))
        n = C.c_int32(0); idx = np.zeros(4, np.uint32); gam, ssq = D(0), D(0)
        ok = self.lib.orc_ut_search(self.ctx, _p(v, D), D(q0), _p(uo, C.c_uint32), _p(ux, self.creal),
                                    _p(ul, self.creal), _p(uh, self.creal), C.byref(n), _p(idx, C.c_uint32),
                                    C.byref(gam), C.byref(ssq))
        return dict(ok=bool(ok), n=n.value, idx=idx, gamma=gam.value, ssq=ssq.value)
