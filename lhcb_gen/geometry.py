"""Default toy geometry and tunables: the *inputs* of ``lhcb_geom_init``.

This module holds numbers only (the paper's printed constants plus the readings
DESIGN.md lists for what the paper leaves open).  It contains none of the
method's arithmetic: both the oracle binding and the CUDA binding marshal this
dictionary into their own, separately declared structs.

Units: mm, MeV/c, q/p in 1/MeV, slopes dimensionless.
Citations are PAPER.md line numbers / equations.
"""
from __future__ import annotations

import copy
import math

TAN5 = math.tan(math.radians(5.0))

# three stations, four layers each, x-u-v-x, stereo +5 (u) / -5 (v) deg.
# z positions: BASELINE.json configs[0].
SCIFI_Z = [7826.0, 7896.0, 7966.0, 8036.0,
           8508.0, 8578.0, 8648.0, 8718.0,
           9193.0, 9263.0, 9333.0, 9403.0]
SCIFI_TAN = [0.0, +TAN5, -TAN5, 0.0] * 3
X_LAYERS = [0, 3, 4, 7, 8, 11]
UV_LAYERS = [1, 2, 5, 6, 9, 10]

DEFAULT_GEOM = {
    # --- SciFi geometry ---------------------------------------------------
    "scifi_z": SCIFI_Z,
    "scifi_tan_alpha": SCIFI_TAN,
    "z_ref": 8525.0,            # Eq. 1
    "d_ratio": -3.3e-4,         # BASELINE.json configs[0] ("b"); paper gives no value (L72)
    # --- XZ seeding windows -------------------------------------------------
    "p_min": 3000.0,            # L78, L90
    "inv_p_a": 1.6322e-7,       # Eq. 6, read per MeV (reading A1)
    "inv_p_b": -5.0217e-12,     # Eq. 6
    "alpha0": 2.180e6,          # Eq. 10
    "alpha1": -1073.0,          # Eq. 10
    "iter_layers": [[0, 4, 8], [3, 7, 11]],   # reading A5 (L78: disjoint triples)
    "kappa_cx": 0.03,           # cx = polarity*q*kappa/p  (reading A3; MeV/mm)
    "cx_band": [0.5, 1.8, 1.0e-6, 1.0e-6],    # f_lo, f_hi, d_lo, d_hi (reading A4, Fig. 6)
    "tol_x_ext": 1.0,           # L90
    "tol_uv": 2.0,              # L215
    "min_x_hits": 5,            # L90
    "min_uv_hits": 4,           # reading A9
    "uv_first_layer": [1, 6],   # reading A9
    "sigma_hit": 0.080,         # BASELINE.json configs[0] sigma_x (reading A6)
    "chi2x_max": 8.0,           # reading A6
    "chi2y_max": 8.0,           # reading A6
    "y_min": -2500.0,           # BASELINE.json configs[1]
    "y_max": 2500.0,
    "y_half_tol": 5.0,          # L372: halves overlap slightly for the first-layer window
    # --- matching ------------------------------------------------------------
    "z_velo": 770.0,            # BASELINE.json configs[1]
    "z_scifi_state": 7826.0,    # BASELINE.json configs[4]
    "z_match_y": 10000.0,       # L231
    "mag": [5287.6, -7.98878, 317.683, 0.0119379, -1418.42],   # Table 1
    "gamma_ab": [7.707063e-11, -7.817364e-3],                  # Table 1
    "kick_pt": 1100.0,          # K_B, MeV (reading A10)
    "polarity": -1,             # +1 magnet up / -1 magnet down (L33)
    "presel": [20.0, 150.0, 1.5, 0.02],                        # Eq. 21
    # Eq. 23: 4/5, 10.12, 101.0, 1/5, 1.59, 212.1, tol_tx = 1/2, 1/tol_ty = 937.5
    "match_tol": [0.8, 10.12, 101.0, 0.2, 1.59, 212.1, 0.5, 937.5],
    "chi2_match_max": 2.0,      # L301
    # --- UT -------------------------------------------------------------------
    "ut_z": [2327.0, 2372.0, 2597.0, 2642.0],                  # BASELINE.json configs[1]
    "ut_tan_alpha": [0.0, +TAN5, -TAN5, 0.0],                  # UTaX, UTaU, UTbV, UTbX (L315)
    # Table 2 (L323-340): A, B (mm*GeV -> multiplies 1/p in 1/GeV), min, max per layer.
    # UTbX loose row is garbled: reading A12.  UTaX tight is unused (first layer always loose):
    # filled with the UTaU values.
    "ut_loose": [[0.8333, 3.3333, 1.2, 8.5],
                 [0.8333, 3.3333, 1.2, 8.5],
                 [1.3333, 3.3333, 1.5, 9.5],
                 [1.5555, 3.3333, 1.5, 9.5]],
    "ut_tight": [[0.2, 0.6, 0.5, 2.0],
                 [0.2, 0.6, 0.5, 2.0],
                 [0.4, 1.2, 1.0, 4.0],
                 [0.4, 1.2, 1.0, 4.0]],
    "ut_y_tol": 1.0,            # DESIGN.md O13
    "ut_strip_x0": -4474 * 0.190,   # strip s sits at x0 = ut_strip_x0 + s * ut_strip_pitch; 8,949 strips over |x| < 850 mm
    "ut_strip_pitch": 0.190,        # L315 / BASELINE.json configs[1]: 190 um pitch
    "ut_row_y0": -700.0,        # UT strips come in 14 sensor rows of 100 mm over |y| < 700 mm (BASELINE.json configs[1])
    "ut_row_pitch": 100.0,
    "min_ut_hits": 3,           # L311 ("more than two")
    "ut_enabled": 1,
    # --- capacities (per event-half / per event); 0 = library default (include/lhcb.h) ---------
    "max_seeds_per_half": 0,
    "max_xz_cand_per_half": 0,
    "max_long_per_event": 0,
    "max_hits_per_half": 0,
    "max_triplets_per_half": 0,
    "max_match_cand_per_event": 0,
    "max_velo_per_event": 0,
    "max_ut_per_event": 0,
}


def default_geom(**overrides):
    """A deep copy of DEFAULT_GEOM with keyword overrides applied."""
    g = copy.deepcopy(DEFAULT_GEOM)
    for k, v in overrides.items():
        if k not in g:
            raise KeyError(f"unknown geometry field {k!r}")
        g[k] = v
    return g
