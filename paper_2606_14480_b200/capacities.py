"""Per-CTA capacities (`lhcb_geom_t.max_*`) for the occupancy of the workload.

All intermediates of both kernels live in shared memory, so the capacities decide how many CTAs share
an SM (include/lhcb.h: lhcb_launch_config).  The library defaults (all zero in the geometry) are sized
for BASELINE.json configs[3] (mu = 7.6 plus displaced tracks); NOMINAL is sized for Run 3 nominal
occupancy (mu ~ 5: configs[1] and configs[2]), where it lets five 256-thread seeding CTAs and six
128-thread matching CTAs share an SM.  Exceeding a capacity is never silent: the per-half / per-event
status words report it and the tests and bench.py fail on any set bit.

Observed maxima over the 16,384 events of configs[2] (seed 2), per event-half: 2,534 hits, 1,144
three-hit combinations per iteration (the queue holds both iterations), 432 x-z candidates, 138 clone-kill survivors, 135 seeds; per
event: 163 VELO states, 3,639 UT hits, 150 chi2-accepted pairs, 166 UT hypotheses.
"""
NOMINAL = dict(max_hits_per_half=2944, max_xz_cand_per_half=512, max_triplets_per_half=2304,
               max_seeds_per_half=192, max_long_per_event=256, max_match_cand_per_event=192,
               max_velo_per_event=192, max_ut_per_event=3840)

# The Hough-cluster UV version (lhcb_set_uv_hough) keeps 136 bytes of tables per clone-kill survivor and queues
# up to 32 hypotheses per survivor: it needs a larger work region than the iterative default, at four CTAs per SM.
NOMINAL_HOUGH = dict(NOMINAL, max_triplets_per_half=4608)


def with_capacities(geom: dict, caps: dict = NOMINAL) -> dict:
    g = dict(geom)
    g.update(caps)
    return g
