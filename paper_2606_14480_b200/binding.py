"""Thin ctypes binding of include/lhcb.h.  Argument marshalling only: every step of the path runs
in the CUDA library.  PyTorch provides device memory and streams.

There is no CPU fallback: importing works without a GPU (so the ABI can be checked), but creating a
Context raises if the library or a CUDA device is missing.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import build as _build

F, I = C.c_float, C.c_int32
NO_HIT = 0xFFFFFFFF
STATIC_MAX_EVENTS = 3072        # LHCB_STATIC_MAX_EVENTS of include/lhcb.h

ST_BITS = {1: "triplet_overflow", 2: "cand_overflow", 4: "seed_overflow", 8: "hits_overflow",
           16: "match_overflow", 32: "long_overflow", 64: "velo_overflow", 128: "ut_overflow", 256: "uv_queue_overflow", 512: "bad_raw_hit"}

EXPORTS = ["lhcb_geom_derive", "lhcb_geom_init", "lhcb_destroy", "lhcb_get_geom", "lhcb_workspace_bytes",
           "lhcb_seeding", "lhcb_matching", "lhcb_error_string", "lhcb_last_cuda_error",
           "lhcb_last_launch_count", "lhcb_pipeline_create", "lhcb_pipeline_destroy", "lhcb_reconstruct_host",
           "lhcb_pipeline_last_bytes", "lhcb_launch_config", "lhcb_prepare", "lhcb_set_ghost_nn", "lhcb_set_uv_hough",
           "lhcb_order", "lhcb_seeding_static"]


class LhcbGeom(C.Structure):
    _fields_ = [
        ("scifi_z", F * 12), ("scifi_tan_alpha", F * 12), ("z_ref", F), ("d_ratio", F),
        ("p_min", F), ("inv_p_a", F), ("inv_p_b", F), ("alpha0", F), ("alpha1", F),
        ("iter_layers", (I * 3) * 2), ("kappa_cx", F), ("cx_band", F * 4),
        ("tol_x_ext", F), ("tol_uv", F), ("min_x_hits", I), ("min_uv_hits", I), ("uv_first_layer", I * 2),
        ("sigma_hit", F), ("chi2x_max", F), ("chi2y_max", F), ("y_min", F), ("y_max", F), ("y_half_tol", F),
        ("z_velo", F), ("z_scifi_state", F), ("z_match_y", F), ("mag", F * 5), ("gamma_ab", F * 2),
        ("kick_pt", F), ("polarity", I), ("presel", F * 4), ("match_tol", F * 8), ("chi2_match_max", F),
        ("ut_z", F * 4), ("ut_tan_alpha", F * 4), ("ut_loose", (F * 4) * 4), ("ut_tight", (F * 4) * 4),
        ("ut_y_tol", F), ("ut_strip_x0", F), ("ut_strip_pitch", F), ("ut_row_y0", F), ("ut_row_pitch", F), ("min_ut_hits", I), ("ut_enabled", I),
        ("max_seeds_per_half", I), ("max_xz_cand_per_half", I), ("max_long_per_event", I),
        ("max_hits_per_half", I), ("max_triplets_per_half", I), ("max_match_cand_per_event", I),
        ("max_velo_per_event", I), ("max_ut_per_event", I),
    ]


class LhcbDerived(C.Structure):
    _fields_ = [
        ("xl", I * 6), ("ul", I * 6), ("slot_of_layer", I * 12),
        ("zb", F * 12), ("gz", F * 12), ("tan_a", F * 12), ("inv_tan", F * 12), ("inv_z", F * 12), ("zt", F * 12),
        ("ywin_a", (F * 12) * 2), ("ywin_b", (F * 12) * 2), ("l1", I * 2), ("l2", I * 2), ("l3", I * 2),
        ("dx3max", F * 2), ("alpha_corr", F * 2), ("r13", F * 2), ("inv_dz13", F * 2), ("z1", F * 2),
        ("dz12", F * 2), ("K", F * 2), ("inv_K", F * 2), ("G13", F * 2),
        ("a", F), ("b", F), ("kappa", F), ("inv_kappa", F), ("f_lo", F), ("f_hi", F), ("d_lo", F), ("d_hi", F),
        ("tol_x", F), ("tol_uv", F), ("chi2x_max", F), ("chi2y_max", F), ("wx", F * 7), ("wy", F * 7),
        ("zbS", F), ("gS", F), ("gpS", F),
        ("zS", F), ("zV", F), ("dzyS", F), ("dzyV", F), ("mag", F * 5), ("presel", F * 4),
        ("cx0", F), ("cx1", F), ("cy0", F), ("cy1", F), ("inv_tol_tx", F), ("inv_tol_ty", F), ("chi2m_max", F),
        ("inv_KB", F), ("Ag", F), ("Bg", F), ("inv_Bg", F), ("ut_dz", F * 4), ("ut_dz2", F * 4), ("ut_dz4", F * 4),
        ("ut_tan", F * 4), ("ut_y_tol", F), ("ut_loose", (F * 4) * 4), ("ut_tight", (F * 4) * 4),
        ("P", ((F * 6) * 3) * 7), ("Q", ((F * 6) * 2) * 64),
    ]


VP = C.c_void_p


class LhcbEvents(C.Structure):
    _fields_ = [("n_events", I), ("n_hits", C.c_uint32), ("zone_off", VP), ("hit_x", VP), ("polarity", VP)]


class LhcbRaw(C.Structure):
    _fields_ = [("n_events", I), ("n_hits", C.c_uint32), ("off", VP), ("x", VP), ("zone", VP)]


class LhcbSeeds(C.Structure):
    _fields_ = [("n_events", I), ("count", VP), ("state", VP), ("par", VP), ("hits", VP), ("nx", VP),
                ("nuv", VP), ("status", VP)]


class LhcbVelo(C.Structure):
    _fields_ = [("n_events", I), ("off", VP), ("x", VP), ("y", VP), ("tx", VP), ("ty", VP), ("polarity", VP)]


class LhcbUt(C.Structure):
    _fields_ = [("n_hits", C.c_uint32), ("off", VP), ("x0", VP), ("y_lo", VP), ("y_hi", VP), ("row", VP), ("strip", VP)]


class LhcbLong(C.Structure):
    _fields_ = [("count", VP), ("seed_idx", VP), ("velo_idx", VP), ("ut_idx", VP), ("n_ut", VP), ("qop", VP),
                ("chi2", VP), ("status", VP), ("ghost", VP)]


class LhcbHostSeeds(C.Structure):
    _fields_ = [("cap", C.c_uint32), ("n", C.c_uint32), ("off", VP), ("state", VP), ("hits", VP), ("nx", VP), ("nuv", VP),
                ("par", VP), ("status", VP)]


class LhcbHostLong(C.Structure):
    _fields_ = [("cap", C.c_uint32), ("n", C.c_uint32), ("off", VP), ("seed_idx", VP), ("velo_idx", VP), ("ut_idx", VP),
                ("n_ut", VP), ("qop", VP), ("chi2", VP), ("status", VP)]


def fill_geom(geom: dict) -> LhcbGeom:
    g = LhcbGeom()
    for name, _ in LhcbGeom._fields_:
        v = geom.get(name, 0)
        if isinstance(v, (list, tuple)):
            arr = getattr(g, name)
            for i, vi in enumerate(v):
                if isinstance(vi, (list, tuple)):
                    for j, vj in enumerate(vi):
                        arr[i][j] = vj
                else:
                    arr[i] = vi
        else:
            setattr(g, name, v)
    return g


_LIB = None


def load_library(build: bool = True, stage_clocks: bool = False, checked: bool = False) -> C.CDLL:
    """dlopen the in-tree library (building it first if the sources are newer).  stage_clocks=True / checked=True
    select a diagnostic build (per-stage cycle counters / index checks); it must be the first load of the process."""
    global _LIB
    if _LIB is None:
        path = _build.build(stage_clocks=stage_clocks, checked=checked) if build else _build.LIB
        if not os.path.exists(path):
            raise RuntimeError(f"CUDA library {path} is missing: run python -m paper_2606_14480_b200.build")
        lib = C.CDLL(path)
        lib.lhcb_geom_derive.argtypes = [C.POINTER(LhcbGeom), C.POINTER(LhcbDerived)]
        lib.lhcb_geom_init.argtypes = [C.POINTER(LhcbGeom), C.c_int, C.POINTER(VP)]
        lib.lhcb_destroy.argtypes = [VP]
        lib.lhcb_destroy.restype = None
        lib.lhcb_get_geom.argtypes = [VP, C.POINTER(LhcbGeom)]
        lib.lhcb_workspace_bytes.argtypes = [VP, C.c_int, C.c_size_t]
        lib.lhcb_workspace_bytes.restype = C.c_size_t
        lib.lhcb_seeding.argtypes = [VP, C.POINTER(LhcbEvents), C.POINTER(LhcbSeeds), VP, VP]
        lib.lhcb_seeding_static.argtypes = [VP, C.POINTER(LhcbEvents), C.POINTER(LhcbSeeds), VP]
        lib.lhcb_matching.argtypes = [VP, C.POINTER(LhcbSeeds), C.POINTER(LhcbVelo), C.POINTER(LhcbUt),
                                      C.POINTER(LhcbLong), VP, VP]
        lib.lhcb_error_string.argtypes = [C.c_int]
        lib.lhcb_error_string.restype = C.c_char_p
        lib.lhcb_last_cuda_error.argtypes = [VP]
        lib.lhcb_last_launch_count.argtypes = [VP]
        lib.lhcb_launch_config.argtypes = [VP, C.POINTER(C.c_int * 4)]
        lib.lhcb_prepare.argtypes = [VP, C.POINTER(LhcbRaw), VP, VP, VP, VP, VP]
        lib.lhcb_set_ghost_nn.argtypes = [VP, C.POINTER(C.c_float)]
        lib.lhcb_set_uv_hough.argtypes = [VP, C.c_int]
        lib.lhcb_order.argtypes = [VP, C.POINTER(LhcbEvents), C.POINTER(LhcbVelo), C.POINTER(LhcbUt), VP, VP]
        lib.lhcb_pipeline_create.argtypes = [VP, C.c_int, C.c_size_t, C.c_size_t, C.c_size_t, C.c_int, C.c_size_t,
                                             C.c_size_t, C.POINTER(VP)]
        lib.lhcb_pipeline_destroy.argtypes = [VP]
        lib.lhcb_pipeline_destroy.restype = None
        lib.lhcb_reconstruct_host.argtypes = [VP, C.POINTER(LhcbEvents), C.POINTER(LhcbVelo), C.POINTER(LhcbUt),
                                              C.POINTER(LhcbHostSeeds), C.POINTER(LhcbHostLong)]
        lib.lhcb_pipeline_last_bytes.argtypes = [VP, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        _LIB = lib
    return _LIB


def lhcb_geom_derive(geom: dict) -> LhcbDerived:
    """Host-only: derived constants of a geometry (no GPU needed)."""
    lib = load_library()
    d = LhcbDerived()
    rc = lib.lhcb_geom_derive(C.byref(fill_geom(geom)), C.byref(d))
    if rc != 0:
        raise ValueError(f"lhcb_geom_derive: {lib.lhcb_error_string(rc).decode()}")
    return d


def _check(lib, ctx, rc, what):
    if rc != 0:
        extra = f" (cudaError {lib.lhcb_last_cuda_error(ctx)})" if rc == -3 and ctx else ""
        raise RuntimeError(f"{what}: {lib.lhcb_error_string(rc).decode()}{extra}")


def _ptr(t):
    return VP(t.data_ptr()) if t is not None else VP(0)


@dataclass
class DeviceEvents:
    """A batch resident in device memory (torch tensors)."""
    n_events: int
    n_hits: int
    zone_off: "torch.Tensor"
    hit_x: "torch.Tensor"
    polarity: Optional["torch.Tensor"]
    velo_off: "torch.Tensor"
    velo_x: "torch.Tensor"
    velo_y: "torch.Tensor"
    velo_tx: "torch.Tensor"
    velo_ty: "torch.Tensor"
    ut_off: Optional["torch.Tensor"] = None
    ut_x0: Optional["torch.Tensor"] = None
    ut_ylo: Optional["torch.Tensor"] = None
    ut_yhi: Optional["torch.Tensor"] = None
    ut_row: Optional["torch.Tensor"] = None     # u8 strip rows: used instead of ut_ylo / ut_yhi when present

    @staticmethod
    def from_host(ev, device="cuda:0"):
        import torch

        def up(a, dt):
            return torch.from_numpy(np.ascontiguousarray(a, dt).view(
                np.int32 if dt == np.uint32 else dt)).to(device)
        has_ut = len(ev.ut_x0) > 0
        return DeviceEvents(
            n_events=ev.n_events, n_hits=ev.n_hits, zone_off=up(ev.zone_off, np.uint32),
            hit_x=up(ev.hit_x, np.float32), polarity=up(ev.polarity, np.int8),
            velo_off=up(ev.velo_off, np.uint32), velo_x=up(ev.velo_x, np.float32),
            velo_y=up(ev.velo_y, np.float32), velo_tx=up(ev.velo_tx, np.float32),
            velo_ty=up(ev.velo_ty, np.float32),
            ut_off=up(ev.ut_off, np.uint32) if has_ut else None,
            ut_x0=up(ev.ut_x0, np.float32) if has_ut else None,
            ut_ylo=up(ev.ut_ylo, np.float32) if has_ut else None,
            ut_yhi=up(ev.ut_yhi, np.float32) if has_ut else None,
            ut_row=up(ev.ut_row, np.uint8) if has_ut and getattr(ev, "ut_row", None) is not None else None)

    def input_bytes(self):
        n = 0
        for t in (self.zone_off, self.hit_x, self.polarity, self.velo_off, self.velo_x, self.velo_y, self.velo_tx,
                  self.velo_ty, self.ut_off, self.ut_x0, self.ut_row if self.ut_row is not None else self.ut_ylo,
                  None if self.ut_row is not None else self.ut_yhi):
            if t is not None:
                n += t.numel() * t.element_size()
        return n


class Context:
    """lhcb_geom_init / lhcb_seeding / lhcb_matching on one CUDA device."""

    def __init__(self, geom: dict, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_14480_b200 needs a CUDA device: there is no CPU fallback")
        self.torch = torch
        self.lib = load_library()
        self.device = device
        self.dev = torch.device("cuda", device)
        torch.cuda.init()
        torch.zeros(1, device=self.dev)                 # make sure the primary context exists
        self._ctx = VP(0)
        rc = self.lib.lhcb_geom_init(C.byref(fill_geom(geom)), device, C.byref(self._ctx))
        _check(self.lib, None, rc, "lhcb_geom_init")
        g = LhcbGeom()
        self.lib.lhcb_get_geom(self._ctx, C.byref(g))
        self.max_seeds = g.max_seeds_per_half
        self.max_long = g.max_long_per_event
        self.geom = geom

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            self.lib.lhcb_destroy(self._ctx)
            self._ctx = VP(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self):
        return VP(self.torch.cuda.current_stream(self.dev).cuda_stream)

    # ------------------------------------------------------------------ outputs
    def alloc_seeds(self, n_events):
        t = self.torch
        cap = n_events * 2 * self.max_seeds
        kw = dict(device=self.dev)
        return dict(n_events=n_events, cap_total=cap,
                    count=t.empty(n_events * 2, dtype=t.int32, **kw), state=t.empty((5, cap), dtype=t.float32, **kw),
                    par=t.empty((7, cap), dtype=t.float32, **kw), hits=t.empty((12, cap), dtype=t.int32, **kw),
                    nx=t.empty(cap, dtype=t.uint8, **kw), nuv=t.empty(cap, dtype=t.uint8, **kw),
                    status=t.empty(n_events * 2, dtype=t.int32, **kw))

    def alloc_long(self, n_events):
        t = self.torch
        cap = n_events * self.max_long
        kw = dict(device=self.dev)
        return dict(n_events=n_events, cap_total=cap, count=t.empty(n_events, dtype=t.int32, **kw),
                    seed_idx=t.empty(cap, dtype=t.int32, **kw), velo_idx=t.empty(cap, dtype=t.int32, **kw),
                    ut_idx=t.empty((4, cap), dtype=t.int32, **kw), n_ut=t.empty(cap, dtype=t.uint8, **kw),
                    qop=t.empty(cap, dtype=t.float32, **kw), chi2=t.empty(cap, dtype=t.float32, **kw),
                    status=t.empty(n_events, dtype=t.int32, **kw), ghost=t.zeros(cap, dtype=t.float32, **kw))

    @staticmethod
    def _seeds_struct(s):
        return LhcbSeeds(s["n_events"], _ptr(s["count"]), _ptr(s["state"]), _ptr(s.get("par")), _ptr(s.get("hits")),
                         _ptr(s.get("nx")), _ptr(s.get("nuv")), _ptr(s.get("status")))

    # ------------------------------------------------------------------ the calls
    def lhcb_prepare(self, raw_off, raw_x, raw_zone, out: Optional[dict] = None, want_perm: bool = True) -> dict:
        """Raw hits (device tensors: int32 view of u32 offsets [n_events+1], float32 x, uint8 zone) ->
        dict(zone_off, hit_x, perm, status) of device tensors in the layout lhcb_seeding reads."""
        t = self.torch
        n_events, n_hits = raw_off.numel() - 1, raw_x.numel()
        if out is None:
            kw = dict(device=self.dev)
            out = dict(zone_off=t.empty(n_events * 24 + 1, dtype=t.int32, **kw), hit_x=t.empty(n_hits, dtype=t.float32, **kw),
                       perm=t.empty(n_hits, dtype=t.int32, **kw) if want_perm else None,
                       status=t.empty(n_events, dtype=t.int32, **kw))
        r = LhcbRaw(n_events, n_hits, _ptr(raw_off), _ptr(raw_x), _ptr(raw_zone))
        rc = self.lib.lhcb_prepare(self._ctx, C.byref(r), _ptr(out["zone_off"]), _ptr(out["hit_x"]), _ptr(out.get("perm")),
                                   _ptr(out["status"]), self._stream())
        _check(self.lib, self._ctx, rc, "lhcb_prepare")
        return out

    def lhcb_order(self, dev: DeviceEvents, workspace=None, use_ut: bool = True):
        """CTA order "heaviest first" of a batch -> the workspace tensor to hand to lhcb_seeding / lhcb_matching."""
        t = self.torch
        nb = int(self.lib.lhcb_workspace_bytes(self._ctx, dev.n_events, 0))
        if workspace is None:
            workspace = t.empty(max(nb, 16), dtype=t.uint8, device=self.dev)
        assert workspace.numel() * workspace.element_size() >= nb
        e = LhcbEvents(dev.n_events, dev.n_hits, _ptr(dev.zone_off), _ptr(dev.hit_x), _ptr(dev.polarity))
        v = LhcbVelo(dev.n_events, _ptr(dev.velo_off), _ptr(dev.velo_x), _ptr(dev.velo_y), _ptr(dev.velo_tx),
                     _ptr(dev.velo_ty), _ptr(dev.polarity))
        u = None
        if use_ut and dev.ut_off is not None:
            u = C.byref(LhcbUt(dev.ut_x0.numel(), _ptr(dev.ut_off), _ptr(dev.ut_x0), _ptr(dev.ut_ylo), _ptr(dev.ut_yhi),
                               _ptr(dev.ut_row)))
        rc = self.lib.lhcb_order(self._ctx, C.byref(e), C.byref(v), u, _ptr(workspace), self._stream())
        _check(self.lib, self._ctx, rc, "lhcb_order")
        return workspace

    def lhcb_seeding(self, dev: DeviceEvents, out: Optional[dict] = None, workspace=None) -> dict:
        out = out if out is not None else self.alloc_seeds(dev.n_events)
        e = LhcbEvents(dev.n_events, dev.n_hits, _ptr(dev.zone_off), _ptr(dev.hit_x), _ptr(dev.polarity))
        s = self._seeds_struct(out)
        rc = self.lib.lhcb_seeding(self._ctx, C.byref(e), C.byref(s), _ptr(workspace), self._stream())
        _check(self.lib, self._ctx, rc, "lhcb_seeding")
        return out

    def lhcb_seeding_static(self, dev: DeviceEvents, out: dict) -> dict:
        """Heaviest-first Seeding with the order tables in the library's built-in device array: for callers that
        may not allocate device memory per batch (see include/lhcb.h).  `out` must come from alloc_seeds(), made
        beforehand: this method allocates nothing either.  At most STATIC_MAX_EVENTS (3,072) events; calls that
        overlap on the GPU race on the shared array."""
        e = LhcbEvents(dev.n_events, dev.n_hits, _ptr(dev.zone_off), _ptr(dev.hit_x), _ptr(dev.polarity))
        s = self._seeds_struct(out)
        rc = self.lib.lhcb_seeding_static(self._ctx, C.byref(e), C.byref(s), self._stream())
        _check(self.lib, self._ctx, rc, "lhcb_seeding_static")
        return out

    def lhcb_matching(self, seeds: dict, dev: DeviceEvents, out: Optional[dict] = None, use_ut: bool = True,
                      workspace=None) -> dict:
        out = out if out is not None else self.alloc_long(dev.n_events)
        s = self._seeds_struct(seeds)
        v = LhcbVelo(dev.n_events, _ptr(dev.velo_off), _ptr(dev.velo_x), _ptr(dev.velo_y), _ptr(dev.velo_tx),
                     _ptr(dev.velo_ty), _ptr(dev.polarity))
        u = None
        if use_ut and dev.ut_off is not None:
            u = C.byref(LhcbUt(dev.ut_x0.numel(), _ptr(dev.ut_off), _ptr(dev.ut_x0), _ptr(dev.ut_ylo), _ptr(dev.ut_yhi),
                               _ptr(dev.ut_row)))
        l = LhcbLong(_ptr(out["count"]), _ptr(out["seed_idx"]), _ptr(out["velo_idx"]), _ptr(out["ut_idx"]),
                     _ptr(out["n_ut"]), _ptr(out["qop"]), _ptr(out["chi2"]), _ptr(out["status"]), _ptr(out.get("ghost")))
        rc = self.lib.lhcb_matching(self._ctx, C.byref(s), C.byref(v), u, C.byref(l), _ptr(workspace), self._stream())
        _check(self.lib, self._ctx, rc, "lhcb_matching")
        return out

    def lhcb_set_uv_hough(self, on: bool):
        """Hough-cluster UV seeding (reading A20) instead of the iterative default."""
        _check(self.lib, self._ctx, self.lib.lhcb_set_uv_hough(self._ctx, 1 if on else 0), "lhcb_set_uv_hough")

    def lhcb_set_ghost_nn(self, nn):
        """nn: 339 float32 (mu, isig, W1, b1, W2, b2, cut, margin) or None (back to the chi2 ranking, A14)."""
        if nn is None:
            rc = self.lib.lhcb_set_ghost_nn(self._ctx, None)
        else:
            a = np.ascontiguousarray(nn, np.float32)
            if a.size != 339:
                raise ValueError("the packed network has 339 values")
            rc = self.lib.lhcb_set_ghost_nn(self._ctx, a.ctypes.data_as(C.POINTER(C.c_float)))
        _check(self.lib, self._ctx, rc, "lhcb_set_ghost_nn")

    def last_launch_count(self):
        return int(self.lib.lhcb_last_launch_count(self._ctx))

    def lhcb_launch_config(self):
        """dict(seed_threads, seed_smem, match_threads, match_smem) selected by this context's capacities."""
        out = (C.c_int * 4)()
        _check(self.lib, self._ctx, self.lib.lhcb_launch_config(self._ctx, C.byref(out)), "lhcb_launch_config")
        return dict(zip(("seed_threads", "seed_smem", "match_threads", "match_smem"), (int(x) for x in out)))

    # ------------------------------------------------------------------ helpers (host views of outputs)
    def seeds_from_states(self, n_events, seed_off, state):
        """Direct seeds (BASELINE.json configs[4]): states [5][n] with per-event offsets -> slot layout.
        Event e's seeds go to half 2e first, then half 2e+1, in input order."""
        t = self.torch
        out = self.alloc_seeds(n_events)
        cap, ms = out["cap_total"], self.max_seeds
        cnt = np.diff(seed_off.astype(np.int64))
        if (cnt > 2 * ms).any():
            raise ValueError("more direct seeds per event than 2*max_seeds_per_half")
        ev = np.repeat(np.arange(n_events), cnt)
        k = np.arange(len(ev)) - np.repeat(seed_off[:-1].astype(np.int64), cnt)
        slot = np.where(k < ms, (2 * ev) * ms + k, (2 * ev + 1) * ms + (k - ms))
        st = np.zeros((5, cap), np.float32)
        st[:, slot] = state
        count = np.zeros(2 * n_events, np.int32)
        count[0::2] = np.minimum(cnt, ms); count[1::2] = np.maximum(cnt - ms, 0)
        out["state"].copy_(t.from_numpy(st)); out["count"].copy_(t.from_numpy(count))
        out["status"].zero_()
        out["nx"].fill_(6); out["nuv"].fill_(6)             # states without hits count as full 12-hit seeds (nHits_SciFi input)
        out["hits"] = None; out["par"] = None               # no hit lists: chi2 ties go to the lower seed index (A21)
        return out, slot

    def seeds_to_host(self, s):
        """Compact host view: per seed event, half, slot, state[5], par[7], hits[12], nx, nuv."""
        cnt = s["count"].cpu().numpy().astype(np.int64)
        ms = self.max_seeds
        half = np.repeat(np.arange(len(cnt)), cnt)
        k = np.arange(len(half)) - np.repeat(np.cumsum(cnt) - cnt, cnt)
        slot = half * ms + k
        st = s["state"].cpu().numpy()[:, slot].T
        par = s["par"].cpu().numpy()[:, slot].T
        hits = s["hits"].cpu().numpy().view(np.uint32)[:, slot].T
        return dict(n=len(slot), event=half // 2, half=half % 2, slot=slot, state=st, par=par, hits=hits,
                    nx=s["nx"].cpu().numpy()[slot], nuv=s["nuv"].cpu().numpy()[slot],
                    status=s["status"].cpu().numpy().view(np.uint32))

    def long_to_host(self, l):
        cnt = l["count"].cpu().numpy().astype(np.int64)
        ml = self.max_long
        ev = np.repeat(np.arange(len(cnt)), cnt)
        k = np.arange(len(ev)) - np.repeat(np.cumsum(cnt) - cnt, cnt)
        slot = ev * ml + k
        g = lambda name: l[name].cpu().numpy()
        return dict(n=len(slot), event=ev, seed=g("seed_idx").view(np.uint32)[slot], velo=g("velo_idx").view(np.uint32)[slot],
                    ut=g("ut_idx").view(np.uint32)[:, slot].T, n_ut=g("n_ut")[slot], qop=g("qop")[slot],
                    chi2=g("chi2")[slot], status=g("status").view(np.uint32),
                    ghost=g("ghost")[slot] if l.get("ghost") is not None else None)


class HostPipeline:
    """lhcb_pipeline_create / lhcb_reconstruct_host: host buffers in, host buffers out (the end-to-end
    path: H2D copies, order, seeding, matching, compaction and D2H copies all inside one C-ABI call)."""

    def __init__(self, ctx: Context, ev, slice_events: int = 2048, use_ut: bool = True, want_par: bool = False,
                 seeds_per_event: int = 256, long_per_event: int = 160, ship_strips: bool = True):
        """ev: a host batch (lhcb_gen.Events-like).  Its arrays are copied once into pinned host memory;
        the pipeline's device buffers are sized for this batch.  seeds_per_event / long_per_event size the dense
        output arrays (LHCB_ERR_CAPACITY if a batch needs more)."""
        import torch
        self.ctx, self.torch = ctx, torch
        self.n_events = n = ev.n_events

        def pin(a, dt):
            a = np.ascontiguousarray(a, dt)
            t = torch.from_numpy(a.view(np.int32) if dt == np.uint32 else a)
            return t.pin_memory() if len(a) else t
        self.h = dict(zone_off=pin(ev.zone_off, np.uint32), hit_x=pin(ev.hit_x, np.float32),
                      polarity=pin(ev.polarity, np.int8), velo_off=pin(ev.velo_off, np.uint32),
                      velo_x=pin(ev.velo_x, np.float32), velo_y=pin(ev.velo_y, np.float32),
                      velo_tx=pin(ev.velo_tx, np.float32), velo_ty=pin(ev.velo_ty, np.float32))
        self.has_ut = use_ut and len(ev.ut_x0) > 0
        if self.has_ut:
            self.h.update(ut_off=pin(ev.ut_off, np.uint32), ut_x0=pin(ev.ut_x0, np.float32), ut_row=pin(ev.ut_row, np.uint8))
            if ship_strips and getattr(ev, "ut_strip", None) is not None:
                self.h["ut_strip"] = pin(ev.ut_strip.view(np.int16), np.int16)
        cs, cl = n * seeds_per_event, n * long_per_event
        z = lambda shape, dt: torch.zeros(shape, dtype=dt).pin_memory()
        self.seeds = dict(cap=cs, off=z(2 * n + 1, torch.int32), state=z((5, cs), torch.float32), hits=z((12, cs), torch.int16),
                          nx=z(cs, torch.uint8), nuv=z(cs, torch.uint8), par=z((7, cs), torch.float32) if want_par else None,
                          status=z(2 * n, torch.int32))
        self.long = dict(cap=cl, off=z(n + 1, torch.int32), seed_idx=z(cl, torch.int32), velo_idx=z(cl, torch.int32),
                         ut_idx=z((4, cl), torch.int32), n_ut=z(cl, torch.uint8), qop=z(cl, torch.float32),
                         chi2=z(cl, torch.float32), status=z(n, torch.int32))
        self._p = VP(0)
        rc = ctx.lib.lhcb_pipeline_create(ctx._ctx, n, ev.n_hits, len(ev.velo_x), len(ev.ut_x0) if self.has_ut else 0,
                                          slice_events, cs, cl, C.byref(self._p))
        _check(ctx.lib, ctx._ctx, rc, "lhcb_pipeline_create")
        h = self.h
        self._ev = LhcbEvents(n, ev.n_hits, _ptr(h["zone_off"]), _ptr(h["hit_x"]), _ptr(h["polarity"]))
        self._velo = LhcbVelo(n, _ptr(h["velo_off"]), _ptr(h["velo_x"]), _ptr(h["velo_y"]), _ptr(h["velo_tx"]),
                              _ptr(h["velo_ty"]), _ptr(h["polarity"]))
        self._ut = LhcbUt(len(ev.ut_x0), _ptr(h["ut_off"]), _ptr(h["ut_x0"]), VP(0), VP(0), _ptr(h["ut_row"]),
                          _ptr(h.get("ut_strip"))) if self.has_ut else None
        s, l = self.seeds, self.long
        self._hs = LhcbHostSeeds(cs, 0, _ptr(s["off"]), _ptr(s["state"]), _ptr(s["hits"]), _ptr(s["nx"]), _ptr(s["nuv"]),
                                 _ptr(s["par"]), _ptr(s["status"]))
        self._hl = LhcbHostLong(cl, 0, _ptr(l["off"]), _ptr(l["seed_idx"]), _ptr(l["velo_idx"]), _ptr(l["ut_idx"]),
                                _ptr(l["n_ut"]), _ptr(l["qop"]), _ptr(l["chi2"]), _ptr(l["status"]))

    def lhcb_reconstruct_host(self):
        """One end-to-end pass; returns (h2d_bytes, d2h_bytes, kernel launches).  Results: seeds_to_host(), long_to_host()."""
        lib = self.ctx.lib
        rc = lib.lhcb_reconstruct_host(self._p, C.byref(self._ev), C.byref(self._velo),
                                       C.byref(self._ut) if self._ut is not None else None, C.byref(self._hs), C.byref(self._hl))
        _check(lib, self.ctx._ctx, rc, "lhcb_reconstruct_host")
        a, b = C.c_uint64(0), C.c_uint64(0)
        launches = lib.lhcb_pipeline_last_bytes(self._p, C.byref(a), C.byref(b))
        return a.value, b.value, launches

    def seeds_to_host(self):
        """Dense seeds of the last pass in the form of Context.seeds_to_host (slot = dense index)."""
        s, n = self.seeds, int(self._hs.n)
        off = s["off"].numpy().view(np.uint32).astype(np.int64)
        half = np.repeat(np.arange(2 * self.n_events), np.diff(off))
        return dict(n=n, event=half // 2, half=half % 2, slot=np.arange(n), state=s["state"].numpy()[:, :n].T.copy(),
                    par=s["par"].numpy()[:, :n].T.copy() if s["par"] is not None else None,
                    hits=self._global_hits(s["hits"].numpy().view(np.uint16)[:, :n].T, half), nx=s["nx"].numpy()[:n].copy(),
                    nuv=s["nuv"].numpy()[:n].copy(), status=s["status"].numpy().view(np.uint32).copy(), off=off)

    def _global_hits(self, local, half):
        """Zone-local u16 hit indices [n][12] of the dense seeds -> global u32 indices (LHCB_NO_HIT kept)."""
        zo = self.h["zone_off"].numpy().view(np.uint32).astype(np.int64)
        base = zo[half[:, None] * 12 + np.arange(12)[None, :]]
        return np.where(local == 0xFFFF, NO_HIT, base + local.astype(np.int64)).astype(np.uint32)

    def long_to_host(self):
        l, n = self.long, int(self._hl.n)
        off = l["off"].numpy().view(np.uint32).astype(np.int64)
        ev = np.repeat(np.arange(self.n_events), np.diff(off))
        g = lambda name: l[name].numpy()
        return dict(n=n, event=ev, seed=g("seed_idx").view(np.uint32)[:n].copy(), velo=g("velo_idx").view(np.uint32)[:n].copy(),
                    ut=g("ut_idx").view(np.uint32)[:, :n].T.copy(), n_ut=g("n_ut")[:n].copy(), qop=g("qop")[:n].copy(),
                    chi2=g("chi2")[:n].copy(), status=g("status").view(np.uint32).copy(), ghost=None, off=off)

    def close(self):
        if self._p.value:
            self.ctx.lib.lhcb_pipeline_destroy(self._p)
            self._p = VP(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
