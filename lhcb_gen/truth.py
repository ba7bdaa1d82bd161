"""Truth association and efficiency bookkeeping on generator truth.

A reconstructed seed is associated to a particle if at least `min_purity` of its hits
come from that particle (Ref. 18 of the paper is not
available).  Used identically on oracle output and on CUDA output; it never looks at how
either was computed.
"""
from __future__ import annotations

import numpy as np

NO_HIT = 0xFFFFFFFF


def seed_pids(ev, hits: np.ndarray, min_purity: float = 0.7):
    """hits: u32[n_seeds, 12] global hit indices (NO_HIT if none) -> (pid i32[n], purity f32[n])."""
    n = hits.shape[0]
    pid = np.full(n, -1, np.int32)
    pur = np.zeros(n, np.float32)
    if n == 0:
        return pid, pur
    valid = hits != NO_HIT
    hp = np.where(valid, ev.hit_pid[np.where(valid, hits, 0)], -2)
    nh = valid.sum(1)
    for j in range(hits.shape[1]):          # majority vote: try each column's pid as candidate
        c = hp[:, j]
        cnt = ((hp == c[:, None]) & valid).sum(1)
        better = (c >= 0) & (cnt > pur * nh)
        pid = np.where(better, c, pid)
        pur = np.where(better, cnt / np.maximum(nh, 1), pur).astype(np.float32)
    pid = np.where(pur >= min_purity, pid, -1).astype(np.int32)
    return pid, pur


def reconstructible_seed(ev, p_factor: float = 1.15):
    """Denominator of the seeding efficiency: in acceptance in all 12 layers, one
    detector half, p >= p_factor*p_min, and >=5 x-hits and >=4 stereo hits recorded."""
    P = ev.particles
    return (P["in_acc"] & ~P["half_cross"] & (P["p"] >= p_factor * ev.geom["p_min"])
            & (P["n_x"] >= ev.geom["min_x_hits"]) & (P["n_uv"] >= ev.geom["min_uv_hits"]))


def seeding_summary(ev, hits: np.ndarray):
    """Efficiency / ghost / clone fractions of a seed collection vs generator truth."""
    pid, _ = seed_pids(ev, hits)
    den = reconstructible_seed(ev)
    found = np.zeros(den.shape[0], bool)
    found[pid[pid >= 0]] = True
    n = max(len(pid), 1)
    matched = pid[pid >= 0]
    n_clone = len(matched) - len(np.unique(matched))
    return dict(n_seeds=int(len(pid)), n_reconstructible=int(den.sum()),
                efficiency=float((found & den).sum() / max(den.sum(), 1)),
                ghost_rate=float((pid < 0).sum() / n), clone_rate=float(n_clone / n))


def long_summary(ev, seed_pid_of_track: np.ndarray, velo_idx: np.ndarray):
    """Long-track efficiency vs truth: a long track is correct if its seed's particle equals
    its VELO track's particle."""
    vpid = ev.velo_pid[velo_idx] if len(velo_idx) else np.zeros(0, np.int32)
    good = (seed_pid_of_track >= 0) & (seed_pid_of_track == vpid)
    P = ev.particles
    if "in_acc" in P:
        den = reconstructible_seed(ev) & (P["kind"] == 0)
    else:
        den = P["kind"] == 0
    found = np.zeros(den.shape[0], bool)
    found[seed_pid_of_track[good]] = True
    n = max(len(velo_idx), 1)
    return dict(n_long=int(len(velo_idx)), n_reconstructible=int(den.sum()),
                efficiency=float((found & den).sum() / max(den.sum(), 1)),
                ghost_rate=float((~good).sum() / n))
