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
