"""Algorithmic work model used for the ALU roofline.

`achieved` = algorithmic lane-operations per launch / kernel time, NOT executed instructions.  The
lane-operation count of one event is  sum_k counter_k * unit_cost_k  with the unit costs of SURVEY.md
section 8(d) and the per-event step counters of the workload.  The counters below are the means the CPU
oracle counted on the first 1024 events of BASELINE.json configs[2] (cfg3, seed 2); bench.py's
cpu_baseline leg re-counts them live on its sample and prints them next to these.

peak = 148 SMs x 128 FP32/INT lanes x SM clock (B200_PROFILING.md: 148 SMs, 1965 MHz max) -- one
lane-operation per lane per clock (an FMA counts as one lane-operation here).
"""
import math

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the 16,384-event cfg3 batch, from the
# `ncu --set full` capture summarised in profiles/ (the bench cannot measure DRAM traffic itself)
NCU_DRAM_BYTES_PER_LAUNCH = {"seeding_kernel": 273.247488e6 + 250.793472e6, "matching_kernel": 372.664320e6 + 47.819776e6}
NCU_DRAM_SOURCE = "profiles/r3_ncu_full.md"

N_SM = 148
LANES_PER_SM = 128

# per-event means, cfg3 (nominal occupancy), counted by the oracle's step counters
CFG3_COUNTERS = dict(t1_hits=639.65, pairs=12658.35, triplets=1826.11, ext_ok=477.0, uv_first=2820.54,
                     y_fits=447.37, sv_pairs=21157.16, ut_steps=457.05)
CFG3_MEAN_ZONE = 158.3       # SciFi hits per (half, layer) zone
CFG3_MEAN_UT_ZONE = 867.7    # UT hits per (event, layer)


def lane_ops(counters: dict, mean_zone: float = CFG3_MEAN_ZONE, mean_ut_zone: float = CFG3_MEAN_UT_ZONE):
    """(seeding, matching) algorithmic lane-operations per event from step counters per event."""
    lg = math.ceil(math.log2(max(mean_zone, 2.0)))
    lgu = math.ceil(math.log2(max(mean_ut_zone, 2.0)))
    seeding = (counters["t1_hits"] * (4 + 2 * lg)         # window of Eq. 11: 2 flops + 2 searches
               + counters["pairs"] * (18 + 2 * lg)        # Eq. 3-5, 12 + band + 2 searches
               + counters["triplets"] * (40 + 3 * lg)     # parabola + 3 predictions + 3 searches
               + counters["ext_ok"] * 100                 # least squares + chi2
               + counters["uv_first"] * 5 * (8 + lg)      # 5 stereo layers: predict + search
               + counters["y_fits"] * 60)
    matching = counters["sv_pairs"] * 45 + counters["ut_steps"] * (15 + lgu)
    return seeding, matching


def smem_probe_loads(counters: dict, mean_zone: float = CFG3_MEAN_ZONE):
    """Algorithmic 4-byte shared-memory loads of the Seeding per event (third roofline row), under
    the same binary-search model as lane_ops: a search costs ceil(log2 zone) probes, a window costs the hits it
    holds.  Per T1 hit its x and two searches (Eq. 11); per pair the T3 hit and two searches (band of Eq. 12-14);
    per triplet the T2 hit and three closest-hit searches (+-1 mm, one more load for the neighbour compared);
    per first-layer stereo hit its x and five closest-hit searches (+-2 mm)."""
    lg = math.ceil(math.log2(max(mean_zone, 2.0)))
    return (counters["t1_hits"] * (1 + 2 * lg) + counters["pairs"] * (1 + 2 * lg)
            + counters["triplets"] * (1 + 3 * (lg + 1)) + counters["uv_first"] * (1 + 5 * (lg + 1)))


def smem_peak(sm_mhz: float) -> float:
    """bytes per second: 148 SMs x 128 B per clock (32 banks x 4 B) x SM clock."""
    return N_SM * 128 * sm_mhz * 1e6


def alu_peak(sm_mhz: float) -> float:
    """lane-operations per second at the given SM clock."""
    return N_SM * LANES_PER_SM * sm_mhz * 1e6


def hbm_bytes_per_event(n_hits, n_velo, n_ut_probes, n_seeds, n_long):
    """Algorithmic DRAM bytes of one event: hits read once, VELO read once, 32 B per UT
    probe, seeds written + read (state only is read back), long tracks written."""
    return 4 * n_hits + 100 + 16 * n_velo + 32 * n_ut_probes + n_seeds * (98 + 20) + n_long * 33
