"""Seeded synthetic inputs + default geometry + truth bookkeeping.

Shared by the oracle tests and the CUDA tests/bench.  Holds none of the
reconstruction arithmetic.
"""
from .geometry import DEFAULT_GEOM, default_geom, X_LAYERS, UV_LAYERS, TAN5
from .events import GenConfig, Events, config, generate, slice_events
from . import truth
from .raw import shuffle_raw
from .ghost_nn import ghost_nn

__all__ = ["DEFAULT_GEOM", "default_geom", "X_LAYERS", "UV_LAYERS", "TAN5",
           "GenConfig", "Events", "config", "generate", "slice_events", "truth", "shuffle_raw", "ghost_nn"]
