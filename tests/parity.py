"""Comparison of CUDA results with oracle results (used by the -m gpu tests and smoke())."""
import numpy as np

NO_HIT = 0xFFFFFFFF


def seed_keys(event, half, hits, state=None):
    """(event, half, 12 hit indices): the identity of a seed (`state` is accepted and ignored)."""
    return [(int(e), int(h)) + tuple(int(x) for x in row) for e, h, row in zip(event, half, hits)]


def compare_seeds(orc, gpu, rtol=1e-4, x_atol=5e-3):
    """orc: Oracle.seeding() dict; gpu: Context.seeds_to_host() dict.
    Returns dict(n_orc, n_gpu, n_common, only_orc, only_gpu, max_rel, max_dx)."""
    ko = seed_keys(orc["event"], orc["half"], orc["hits"])
    kg = seed_keys(gpu["event"], gpu["half"], gpu["hits"])
    io = {k: i for i, k in enumerate(ko)}
    ig = {k: i for i, k in enumerate(kg)}
    assert len(io) == len(ko), "duplicate seeds in oracle output"
    assert len(ig) == len(kg), "duplicate seeds in CUDA output"
    common = [k for k in ko if k in ig]
    a = np.array([io[k] for k in common], np.int64); b = np.array([ig[k] for k in common], np.int64)
    res = dict(n_orc=len(ko), n_gpu=len(kg), n_common=len(common),
               only_orc=[k for k in ko if k not in ig], only_gpu=[k for k in kg if k not in io],
               max_rel=0.0, max_dx=0.0, bit_equal=True)
    if len(common):
        so, sg = orc["state"][a].astype(np.float64), gpu["state"][b].astype(np.float64)
        po, pg = orc["par"][a].astype(np.float64), gpu["par"][b].astype(np.float64)
        res["bit_equal"] = bool(np.array_equal(orc["state"][a].astype(np.float32).view(np.uint32),
                                               gpu["state"][b].view(np.uint32))
                                and np.array_equal(orc["par"][a].astype(np.float32).view(np.uint32),
                                                   gpu["par"][b].view(np.uint32)))
        res["max_dx"] = float(np.abs(so[:, 0] - sg[:, 0]).max())
        floors = np.array([1e-3, 1e-6, 1e-7, 1e-3, 1e-6, 1e-3, 1e-3])       # ax bx cx ay by chi2x chi2y
        rel = np.abs(po - pg) / np.maximum(np.abs(po), floors)
        res["max_rel"] = float(rel.max())
        assert (orc["nx"][a] == gpu["nx"][b]).all() and (orc["nuv"][a] == gpu["nuv"][b]).all()
    return res


def long_keys(m, seed_key_of):
    return [(seed_key_of[int(s)], int(v)) + tuple(int(x) for x in u) for s, v, u in zip(m["seed"], m["velo"], m["ut"])]


def compare_long(orc_m, gpu_m, orc_seed_key, gpu_seed_key):
    """Long tracks as sets of (seed identity, velo index, UT hit indices)."""
    ko = long_keys(orc_m, orc_seed_key); kg = long_keys(gpu_m, gpu_seed_key)
    io = {k: i for i, k in enumerate(ko)}; ig = {k: i for i, k in enumerate(kg)}
    assert len(io) == len(ko) and len(ig) == len(kg)
    # strict: since reading A21 (exact chi2 ties between twin seeds are decided by their hit lists) the set of
    # long tracks is unique, whatever the order in which the seeds were written
    common = [(k, k) for k in ko if k in ig]
    only_orc = [k for k in ko if k not in ig]; only_gpu = [k for k in kg if k not in io]
    a = np.array([io[k] for k, _ in common], np.int64); b = np.array([ig[g] for _, g in common], np.int64)
    res = dict(n_orc=len(ko), n_gpu=len(kg), n_common=len(common), only_orc=only_orc, only_gpu=only_gpu,
               max_rel_qop=0.0, max_rel_chi2=0.0, bit_equal=True, pairs=(a, b))
    if len(common):
        qo, qg = orc_m["qop"][a].astype(np.float64), gpu_m["qop"][b].astype(np.float64)
        co, cg = orc_m["chi2"][a].astype(np.float64), gpu_m["chi2"][b].astype(np.float64)
        res["max_rel_qop"] = float((np.abs(qo - qg) / np.maximum(np.abs(qo), 1e-9)).max())
        res["max_rel_chi2"] = float((np.abs(co - cg) / np.maximum(np.abs(co), 1e-6)).max())
        res["bit_equal"] = bool(np.array_equal(orc_m["qop"][a].astype(np.float32).view(np.uint32), gpu_m["qop"][b].view(np.uint32))
                                and np.array_equal(orc_m["chi2"][a].astype(np.float32).view(np.uint32), gpu_m["chi2"][b].view(np.uint32)))
        assert (orc_m["n_ut"][a] == gpu_m["n_ut"][b]).all()
    return res


# ---------------------------------------------------------------------------------------- whole batches
def _seed_matrix(s):
    return np.column_stack([np.asarray(s["event"], np.int64), np.asarray(s["half"], np.int64), s["hits"].astype(np.int64)])


def assert_batch_identical(orc_s, orc_m, gpu_s, gpu_m, what=""):
    """Whole-batch, vectorised: the CUDA seeds and long tracks equal the oracle's as sets, with bit-identical
    float32 parameters.  gpu_m["seed"] refers to gpu_s["slot"]; orc_m["seed"] to the row of orc_s.
    Returns (n_seeds, n_long)."""
    ko, kg = _seed_matrix(orc_s), _seed_matrix(gpu_s)
    oo, og = np.lexsort(ko.T[::-1]), np.lexsort(kg.T[::-1])
    assert ko.shape == kg.shape, (what, "seed counts differ", ko.shape, kg.shape)
    assert np.array_equal(ko[oo], kg[og]), (what, "seed hit sets differ")
    assert len(np.unique(ko, axis=0)) == len(ko), (what, "duplicate seeds")
    for name in ("state", "par"):
        a = np.ascontiguousarray(orc_s[name][oo], np.float32).view(np.uint32)
        b = np.ascontiguousarray(gpu_s[name][og], np.float32).view(np.uint32)
        assert np.array_equal(a, b), (what, name, "not bit-identical")
    assert np.array_equal(orc_s["nx"][oo], gpu_s["nx"][og]) and np.array_equal(orc_s["nuv"][oo], gpu_s["nuv"][og])
    # long tracks: (seed identity, velo, ut hits)
    slot_sorted = np.argsort(gpu_s["slot"])
    row_of_slot = slot_sorted[np.searchsorted(gpu_s["slot"][slot_sorted], gpu_m["seed"].astype(np.int64))]
    lo = np.column_stack([ko[orc_m["seed"].astype(np.int64)], orc_m["velo"].astype(np.int64), orc_m["ut"].astype(np.int64)])
    lg = np.column_stack([kg[row_of_slot], gpu_m["velo"].astype(np.int64), gpu_m["ut"].astype(np.int64)])
    po, pg = np.lexsort(lo.T[::-1]), np.lexsort(lg.T[::-1])
    assert lo.shape == lg.shape, (what, "long-track counts differ", lo.shape, lg.shape)
    assert np.array_equal(lo[po], lg[pg]), (what, "long tracks differ")
    names = ("qop", "chi2") + (("ghost",) if "ghost" in orc_m and gpu_m.get("ghost") is not None else ())
    for name in names:
        a = np.ascontiguousarray(orc_m[name][po], np.float32).view(np.uint32)
        b = np.ascontiguousarray(gpu_m[name][pg], np.float32).view(np.uint32)
        assert np.array_equal(a, b), (what, name, "not bit-identical")
    assert np.array_equal(orc_m["n_ut"][po], gpu_m["n_ut"][pg])
    return len(ko), len(lo)


def select_events(s, m, keep_event, slot_key="slot"):
    """Rows of a seeds dict / long-track dict whose event is flagged in keep_event (bool per event)."""
    ks = keep_event[np.asarray(s["event"], np.int64)]
    s2 = {k: (v[ks] if isinstance(v, np.ndarray) and v.shape[:1] == ks.shape else v) for k, v in s.items()}
    km = keep_event[np.asarray(m["event"], np.int64)]
    m2 = {k: (v[km] if isinstance(v, np.ndarray) and v.shape[:1] == km.shape else v) for k, v in m.items()}
    if slot_key not in s:                       # oracle: m["seed"] is a row index -> renumber
        new_row = np.cumsum(ks) - 1
        m2["seed"] = new_row[m2["seed"].astype(np.int64)].astype(np.uint32)
    return s2, m2
