"""The oracle on all host cores (TEST INFRASTRUCTURE, like everything under oracle/): N independent
single-threaded oracle processes over contiguous event shards (SURVEY.md 8(d) "Oracle timing": events are
independent), results merged with batch-global indices.  The oracle itself is untouched: each
process calls Oracle.reconstruct (or Oracle.matching for direct seeds) on its shard exactly as a single process
would on the whole batch."""
from __future__ import annotations

import multiprocessing as mp
import os
import time

import numpy as np

NO_HIT = 0xFFFFFFFF
_JOB = {}


def _run(args):
    a, b = args
    from lhcb_gen import slice_events
    from oracle.binding import Oracle
    ev, mode, use_ut, hough, direct = _JOB["ev"], _JOB["mode"], _JOB["use_ut"], _JOB["hough"], _JOB["direct"]
    nn = _JOB.get("nn")
    sub = slice_events(ev, a, b)
    o = Oracle(ev.geom, mode)
    if hough:
        o.set_uv_hough(True)
    t = time.perf_counter()
    if direct:
        s = None
        m = o.matching(sub.n_events, sub.seed_off, sub.seed_state.T, sub, use_ut=use_ut, nn=nn)
    elif nn is not None:                                     # final selection by the ghost network (A14b), on the oracle's own seeds
        s = o.seeding(sub)
        seed_off = np.zeros(sub.n_events + 1, np.uint32)
        np.cumsum(np.bincount(s["event"], minlength=sub.n_events), out=seed_off[1:])
        m = o.matching(sub.n_events, seed_off, s["state"], sub, use_ut=use_ut, nn=nn,
                       nhits=(s["nx"] + s["nuv"]).astype(np.uint8))
    else:
        s, m = o.reconstruct(sub, use_ut=use_ut)
    return a, b, s, m, time.perf_counter() - t


def reconstruct_parallel(ev, workers: int | None = None, mode: str = "f32", use_ut: bool = True, hough: bool = False,
                         direct_seeds: bool = False, shard_events: int | None = None, nn=None):
    """(seeds, long tracks, info) of the whole batch; seeds is None for direct seeds (BASELINE.json configs[4]).
    info: workers, wall seconds, summed CPU seconds, merged step counters.
    nn: the 339 packed values of the ghost-killing network (reading A14b; long tracks then carry "ghost") or None."""
    workers = max(1, workers or os.cpu_count() or 1)
    n = ev.n_events
    shard = shard_events or max(1, -(-n // (workers * 4)))
    jobs = [(a, min(a + shard, n)) for a in range(0, n, shard)]
    _JOB.update(ev=ev, mode=mode, use_ut=use_ut, hough=hough, direct=direct_seeds, nn=nn)
    t0 = time.perf_counter()
    if workers > 1 and len(jobs) > 1:
        with mp.get_context("fork").Pool(min(workers, len(jobs))) as pool:
            parts = pool.map(_run, jobs, chunksize=1)
    else:
        parts = [_run(j) for j in jobs]
    wall = time.perf_counter() - t0
    _JOB.clear()
    parts.sort(key=lambda p: p[0])
    zo, vo, uo = ev.zone_off.astype(np.int64), ev.velo_off.astype(np.int64), ev.ut_off.astype(np.int64)
    seeds, longs, seed_base = [], [], 0
    counters = {}
    for a, b, s, m, _ in parts:
        m = dict(m)
        m["event"] = m["event"] + a
        m["velo"] = (m["velo"].astype(np.int64) + vo[a]).astype(np.uint32)
        u = m["ut"].astype(np.int64)
        m["ut"] = np.where(u == NO_HIT, u, u + (uo[a * 4] if len(uo) > a * 4 else 0)).astype(np.uint32)
        if s is not None:
            s = dict(s)
            s["event"] = s["event"] + a
            h = s["hits"].astype(np.int64)
            s["hits"] = np.where(h == NO_HIT, h, h + zo[a * 24]).astype(np.uint32)
            m["seed"] = (m["seed"].astype(np.int64) + seed_base).astype(np.uint32)
            seed_base += s["n"]
            seeds.append(s)
        else:
            m["seed"] = (m["seed"].astype(np.int64) + int(ev.seed_off[a])).astype(np.uint32)
        longs.append(m)
        for part in (s, m):
            if part is not None:
                for k, v in part["counters"].items():
                    counters[k] = counters.get(k, 0) + v

    def cat(parts_, keys):
        out = {k: np.concatenate([p[k] for p in parts_]) for k in keys}
        out["n"] = int(sum(p["n"] for p in parts_))
        return out
    S = cat(seeds, ["event", "half", "state", "par", "hits", "nx", "nuv"]) if seeds else None
    M = cat(longs, ["event", "seed", "velo", "ut", "n_ut", "qop", "chi2"] + (["ghost"] if nn is not None else []))
    info = dict(workers=min(workers, len(jobs)), wall_s=wall, cpu_s=float(sum(p[4] for p in parts)), counters=counters)
    return S, M, info
