"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol include/lhcb.h
declares, and its host-only constant derivation agrees with the oracle's independent derivation."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from lhcb_gen import default_geom
from paper_2606_14480_b200 import EXPORTS, lhcb_geom_derive, load_library
from paper_2606_14480_b200.binding import LhcbGeom, LhcbDerived, fill_geom

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    lib = load_library()
    header = open(os.path.join(ROOT, "include", "lhcb.h")).read()
    declared = set(re.findall(r"\b(lhcb_[a-z_]+)\s*\(", header))
    assert declared == set(EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_struct_sizes_match_header():
    # sizes implied by the header's field lists (floats/ints are 4 bytes, no padding needed)
    assert C.sizeof(LhcbGeom) == 4 * (12 + 12 + 2 + 5 + 6 + 1 + 4 + 2 + 2 + 2 + 3 + 3 + 3 + 5 + 2 + 1 + 1 + 4 + 8 + 1
                                      + 4 + 4 + 16 + 16 + 1 + 2 + 2 + 2 + 8)
    assert C.sizeof(LhcbDerived) == 4 * (6 + 6 + 12 + 6 * 12 + 2 * 24 + 6 + 9 * 2 + 12 + 14 + 3 + 4 + 5 + 4 + 7 + 4
                                         + 16 + 1 + 32 + 7 * 18 + 64 * 12)


def test_error_paths_without_gpu():
    lib = load_library()
    assert lib.lhcb_error_string(0) == b"ok" and lib.lhcb_error_string(-2) == b"bad geometry"
    assert lib.lhcb_geom_derive(None, None) == -1
    bad = default_geom(); bad["scifi_tan_alpha"] = [0.0] * 12
    with pytest.raises(ValueError):
        lhcb_geom_derive(bad)
    bad = default_geom(iter_layers=[[0, 5, 8], [3, 7, 11]])        # layer 5 is a stereo layer
    with pytest.raises(ValueError):
        lhcb_geom_derive(bad)
    # geometry validation: first stereo layers, UT hit minimum, Eq. 8 domain, half ranges
    for kw in (dict(uv_first_layer=[1, 12]), dict(uv_first_layer=[0, 6]), dict(min_ut_hits=0), dict(min_ut_hits=5),
               dict(p_min=700.0), dict(y_max=-1.0), dict(y_half_tol=-5.0)):
        with pytest.raises(ValueError):
            lhcb_geom_derive(default_geom(**kw))
    assert lib.lhcb_seeding(None, None, None, None, None) == -4
    assert lib.lhcb_last_launch_count(None) == 0


def test_derived_constants_agree_with_oracle(geom, oracle32):
    """Two independent derivations (QR in double here, Gaussian elimination in long double in the
    oracle) give bit-identical float tables: the precondition for bit-exact parity of the fits."""
    d = lhcb_geom_derive(geom)
    c = oracle32.constants()
    for name in ("dx3max", "alpha_corr", "K", "r13"):
        assert np.array_equal(np.array(getattr(d, name)[:], np.float32), c[name].astype(np.float32)), name
    P = np.array([oracle32.pinv_xz(k) for k in range(7)], np.float32)
    Q = np.array([oracle32.pinv_y(k) for k in range(64)], np.float32)
    assert np.array_equal(P.view(np.uint32), np.ctypeslib.as_array(d.P).view(np.uint32))
    assert np.array_equal(Q.view(np.uint32), np.ctypeslib.as_array(d.Q).view(np.uint32))
    # P is a left inverse of the design matrix for each pattern
    zb = np.array(d.zb[:])[list(d.xl)]; gz = np.array(d.gz[:])[list(d.xl)]
    A = np.stack([np.ones(6), zb, gz], 1).astype(np.float64)
    for k in range(7):
        keep = [s for s in range(6) if k != 1 + s]
        Pk = np.ctypeslib.as_array(d.P)[k].astype(np.float64)
        Dg = np.diag([1.0, 700.0, 5e5])          # compare in units where every column of A is O(1)
        assert np.allclose(Dg @ (Pk[:, keep] @ A[keep]) @ np.linalg.inv(Dg), np.eye(3), atol=1e-5)
        if k:
            assert (Pk[:, k - 1] == 0).all()
