"""B200-native (sm_100a) LHCb HLT1 Seeding + Matching hot path (arxiv/paper_2606_14480).

The product is the C-ABI CUDA library declared in include/lhcb.h (sources in csrc/); this package is
its thin Python binding.  There is no CPU fallback.
"""
from . import capacities, shard, workmodel
from .binding import Context, DeviceEvents, HostPipeline, lhcb_geom_derive, load_library, NO_HIT, EXPORTS

__all__ = ["Context", "DeviceEvents", "HostPipeline", "lhcb_geom_derive", "load_library", "NO_HIT", "EXPORTS"]
