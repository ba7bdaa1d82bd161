#!/usr/bin/env python
"""Throughput bench of the Seeding + Matching hot path (BASELINE.json metric: events/s and long tracks/s,
device-timed, 1 B200, + roofline %).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--events E] [--stage-clocks]

A step = one pass of the whole hot path (lhcb_order + lhcb_seeding + lhcb_matching) over one batch of cfg3
events (BASELINE.json configs[2]: nominal-occupancy events, seed 2, batch 16,384) resident in HBM.  Inputs are
~0.8 GB per batch (> the 126 MB L2), so consecutive steps cannot be served from L2.
Multi-GPU: events are independent: each rank processes its own 16,384-event batch, no
collective on the data path (weak scaling).
--stage-clocks: no timing; builds the diagnostic library variant (-DLHCB_STAGE_CLOCKS) and prints where the
cycles of one CTA go, stage by stage (the table under profiles/).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC, UNIT = "seeding_matching_events_per_s", "events/s"


def sample_clocks(stop, out, gpu_index):
    q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
    while not stop.is_set():
        try:
            r = subprocess.run(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=5)
            f = [x.strip() for x in r.stdout.strip().split(",")]
            if len(f) >= 6:
                out.append(f)
        except Exception:
            pass
        stop.wait(0.05)


def clocks_summary(samples):
    if not samples:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
    sm = [float(s[0]) for s in samples if s[0].replace(".", "").isdigit()]
    mx = [float(s[1]) for s in samples if s[1].replace(".", "").isdigit()]
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    reasons = [n for i, n in enumerate(names) if any(s[2 + i].lower().startswith("active") for s in samples)]
    return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
            "reasons": reasons, "samples": len(samples)}


def _per_event(counters, n):
    return {k: round(v / n, 2) for k, v in counters.items() if v}


def oracle_baseline(ev, n_sample, use_ut=True, all_cores=True):
    """The oracle as it stands on the first n_sample events of the workload: single-threaded, and as independent
    single-threaded processes over event shards on all host cores."""
    from lhcb_gen import slice_events
    from oracle.binding import Oracle
    from oracle.parallel import reconstruct_parallel
    sub = slice_events(ev, 0, min(n_sample, ev.n_events))
    n1 = max(1, min(sub.n_events, n_sample // 8))                      # one core: an eighth of the sample
    one = slice_events(sub, 0, n1)
    o = Oracle(ev.geom, "f32")
    t = time.perf_counter()
    s, m = o.reconstruct(one, use_ut=use_ut)
    dt = time.perf_counter() - t
    out = dict(value=n1 / dt, unit=UNIT, cores=1, kind="oracle",
               sample=f"first {n1} events of the cfg3 batch, seeding+matching, single thread, f32 spec mode",
               long_tracks_per_s=m["n"] / dt)
    counters = {**s["counters"], **{k: v for k, v in m["counters"].items() if v}}
    n_cnt = n1
    if all_cores:
        cores = os.cpu_count() or 1
        S, M, info = reconstruct_parallel(sub, workers=cores, use_ut=use_ut)
        out["all_cores"] = dict(value=sub.n_events / info["wall_s"], unit=UNIT, cores=info["workers"], kind="oracle",
                                sample=f"first {sub.n_events} events of the cfg3 batch as {info['workers']} independent "
                                       f"single-threaded oracle processes over event shards",
                                long_tracks_per_s=M["n"] / info["wall_s"], cpu_seconds=info["cpu_s"])
        counters, n_cnt = info["counters"], sub.n_events
    out["counters_per_event"] = _per_event(counters, n_cnt)
    out["counters_events"] = n_cnt
    return out


def run_reference(args, rank, world):
    if rank != 0:
        return
    from lhcb_gen import config, generate
    n = 128
    ev = generate(config(3, n))
    vals = []
    for i in range(args.warmup + args.steps):
        b = oracle_baseline(ev, 8 * n, all_cores=False)               # one core on all n events
        if i >= args.warmup:
            vals.append(b)
    v = float(np.mean([b["value"] for b in vals]))
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * n / v, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"cfg3 (BASELINE.json configs[2]) nominal-occupancy events, seed 2; each step = the "
                                   f"CPU oracle on a bounded sample of {n} events"},
            "cpu_baseline": {**vals[-1], "value": v},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def stage_clocks(args, local_rank):
    """Where the cycles of a CTA go (thread 0's clock between the stage marks, summed over the CTAs of one launch)."""
    import ctypes
    import torch
    from lhcb_gen import config, generate
    from paper_2606_14480_b200 import Context, DeviceEvents, capacities, load_library
    lib = load_library(stage_clocks=True)
    lib.lhcb_debug_stage_clocks.argtypes = [ctypes.POINTER(ctypes.c_ulonglong * 24), ctypes.c_int]
    n = args.events
    ev = generate(config(3, n), workers=8)
    ev.geom.update(capacities.NOMINAL)
    ctx = Context(ev.geom, device=local_rank)
    dev = DeviceEvents.from_host(ev, f"cuda:{local_rank}")
    seeds, longs = ctx.alloc_seeds(n), ctx.alloc_long(n)
    ws = ctx.lhcb_order(dev)
    for _ in range(3):
        ctx.lhcb_seeding(dev, seeds, workspace=ws); ctx.lhcb_matching(seeds, dev, longs, workspace=ws)
    torch.cuda.synchronize()
    buf = (ctypes.c_ulonglong * 24)()
    lib.lhcb_debug_stage_clocks(ctypes.byref(buf), 1)
    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    st = torch.cuda.current_stream()
    e[0].record(st); ctx.lhcb_seeding(dev, seeds, workspace=ws); e[1].record(st)
    ctx.lhcb_matching(seeds, dev, longs, workspace=ws); e[2].record(st)
    torch.cuda.synchronize()
    lib.lhcb_debug_stage_clocks(ctypes.byref(buf), 0)
    v = np.array(list(buf)[:16], np.float64)
    names = ["S0 staging", "S0 bin tables", "S1 T3 windows + item scan", "S1 pair walk", "S2 extension",
             "S2b fit + S3 clone kill + survivors", "S4 first-layer windows + scan", "S4 u/v walk", "S5 y fit + output",
             "M0 VELO sort", "M1 ranges + scan", "M2 pair loop", "M3 UT search", "M4 selection + output", "M3 wait for the UT tile"]
    print(f"# stage clocks, cfg3 batch of {n} events, capacities.NOMINAL, diagnostic build (-DLHCB_STAGE_CLOCKS):")
    print(f"# seeding {e[0].elapsed_time(e[1]):.3f} ms, matching {e[1].elapsed_time(e[2]):.3f} ms in this build")
    print("| kernel | stage | share of the CTA's cycles | cycles per CTA |")
    print("|---|---|---|---|")
    for lo, hi, kern, nct in ((0, 9, "seeding_kernel", 2 * n), (9, 15, "matching_kernel", n)):
        tot = v[lo:hi].sum()
        for i in range(lo, hi):
            if v[i] > 0:
                print(f"| {kern} | {names[i]} | {100 * v[i] / tot:.1f}% | {v[i] / nct:.0f} |")
    print("# maxima over CTAs: triplets %d, x-z candidates %d, survivors %d, u/v combinations %d, accepted pairs %d, UT hypotheses %d"
          % tuple(int(x) for x in list(buf)[16:22]))


def pcie_bandwidth(torch, dev, nbytes=256 << 20):
    """GB/s host->device, device->host (one direction at a time), and of both directions running together (the
    pipeline's steady state: inputs of a slice go in while results of an earlier one come out)."""
    h, h2 = torch.empty(nbytes, dtype=torch.uint8).pin_memory(), torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d, d2 = torch.empty(nbytes, dtype=torch.uint8, device=dev), torch.empty(nbytes, dtype=torch.uint8, device=dev)
    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    best = [0.0, 0.0, 0.0, 0.0]
    for _ in range(3):
        e[0].record(); d.copy_(h, non_blocking=True); e[1].record(); h.copy_(d, non_blocking=True); e[2].record()
        torch.cuda.synchronize()
        best[0] = max(best[0], nbytes / e[0].elapsed_time(e[1]) / 1e6)
        best[1] = max(best[1], nbytes / e[1].elapsed_time(e[2]) / 1e6)
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    a = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    for _ in range(3):
        torch.cuda.synchronize()
        with torch.cuda.stream(s_in):
            a[0].record(); d.copy_(h, non_blocking=True); a[1].record()
        with torch.cuda.stream(s_out):
            a[2].record(); h2.copy_(d2, non_blocking=True); a[3].record()
        torch.cuda.synchronize()
        best[2] = max(best[2], nbytes / a[0].elapsed_time(a[1]) / 1e6)
        best[3] = max(best[3], nbytes / a[2].elapsed_time(a[3]) / 1e6)
    return best


def pcie_replay(torch, dev, h2d_bytes, d2h_bytes, n_slices=10, reps=5):
    """The floor of the end-to-end leg on this box: the same bytes in the same directions at the same time, cut
    into as many copies as the pipeline issues (3 input and 11 output arrays per slice + the batch-wide small
    arrays), pinned memory, no kernels.  Milliseconds per batch, best of reps."""
    h_in, d_in = torch.empty(h2d_bytes, dtype=torch.uint8).pin_memory(), torch.empty(h2d_bytes, dtype=torch.uint8, device=dev)
    h_out, d_out = torch.empty(d2h_bytes, dtype=torch.uint8).pin_memory(), torch.empty(d2h_bytes, dtype=torch.uint8, device=dev)
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    best = float("inf")
    for _ in range(reps):
        torch.cuda.synchronize()
        t = time.perf_counter()
        with torch.cuda.stream(s_in):
            off = 0
            for frac in (0.0033, 0.0001, 0.0002, 0.0172, 0.0172, 0.0172, 0.0172, 0.0006):     # offsets, polarity, VELO
                b = int(h2d_bytes * frac); d_in[off:off + b].copy_(h_in[off:off + b], non_blocking=True); off += b
            per = (h2d_bytes - off) // n_slices
            for _k in range(n_slices):
                for frac in (0.6, 0.27, 0.13):                                               # hits, UT strips, UT rows
                    b = int(per * frac); d_in[off:off + b].copy_(h_in[off:off + b], non_blocking=True); off += b
        with torch.cuda.stream(s_out):
            per, off = d2h_bytes // n_slices, 0
            for _k in range(n_slices):
                for frac in (0.3, 0.36, 0.015, 0.015, 0.06, 0.06, 0.12, 0.01, 0.03, 0.03):     # seed and long-track arrays
                    b = int(per * frac); h_out[off:off + b].copy_(d_out[off:off + b], non_blocking=True); off += b
        torch.cuda.synchronize()
        best = min(best, (time.perf_counter() - t) * 1e3)
    return best


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=16384, help="events per GPU batch (cfg3: 16384)")
    ap.add_argument("--cpu-sample", type=int, default=4096, help="events the oracle is timed on (all cores; one core: an eighth)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--stage-clocks", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.stage_clocks:
        if rank == 0:
            stage_clocks(args, local_rank)
        return

    import torch
    import torch.distributed as dist
    from lhcb_gen import config, generate
    from paper_2606_14480_b200 import Context, DeviceEvents, HostPipeline, capacities, shard, workmodel

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    # ---- workload: cfg3, this rank's own batch --------------------------------------------------
    n = args.events
    first_chunk, _ = shard.weak_chunks(rank, n)              # rank r generates its own chunk range (weak scaling)
    workers = max(1, min(8, (os.cpu_count() or 8) // max(world, 1)))
    ev = generate(config(3, n), workers=workers, first_chunk=first_chunk)
    ev.geom.update(capacities.NOMINAL)                       # per-CTA capacities for nominal occupancy
    ctx = Context(ev.geom, device=local_rank)
    launch = ctx.lhcb_launch_config()
    dev = DeviceEvents.from_host(ev, f"cuda:{local_rank}")
    seeds, longs = ctx.alloc_seeds(n), ctx.alloc_long(n)
    ws = ctx.lhcb_order(dev)
    stream = torch.cuda.current_stream()

    def step(evts=None):
        # (an event recorded between the two kernels would keep the Matching from starting under the tail of the
        # Seeding grid: the timed steps carry none; the per-kernel times come from a separate loop below)
        # returns the kernels launched, as the library counted them (lhcb_order launches none above 3,072 events)
        if evts:
            evts[0].record(stream)
        ctx.lhcb_order(dev, ws); nl = ctx.last_launch_count()
        ctx.lhcb_seeding(dev, seeds, workspace=ws); nl += ctx.last_launch_count()
        if evts:
            evts[1].record(stream)
        ctx.lhcb_matching(seeds, dev, longs, workspace=ws); nl += ctx.last_launch_count()
        if evts:
            evts[2].record(stream)
        return nl

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sh = ctx.seeds_to_host(seeds); lt = ctx.long_to_host(longs)
    if sh["status"].any() or lt["status"].any():
        raise SystemExit("capacity overflow in the bench workload: results would be incomplete")
    n_long = int(lt["n"]); n_seeds = int(sh["n"])

    # ---- timed region: exactly K steps -------------------------------------------------------------
    K = args.steps
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    samples, stop = [], threading.Event()
    th = threading.Thread(target=sample_clocks, args=(stop, samples, local_rank), daemon=True)
    barrier()
    th.start()
    t0.record(stream)
    gpu_launches = 0
    for k in range(K):
        gpu_launches += step()
    t1.record(stream)
    torch.cuda.synchronize()
    stop.set(); th.join()
    total_ms = t0.elapsed_time(t1)
    # per-kernel times (CUDA events between the kernels, on the stream they are launched on)
    evts = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(min(K, 50))]
    for ev3 in evts:
        step(ev3)
    torch.cuda.synchronize()
    total_ms, summed = shard.reduce_report(total_ms, {"long": n_long}, device="cuda")   # max time, summed counters
    n_long_all = summed["long"]
    seed_ms = np.array([e[0].elapsed_time(e[1]) for e in evts]); match_ms = np.array([e[1].elapsed_time(e[2]) for e in evts])
    ms_per_step = total_ms / K
    value = world * n / (ms_per_step * 1e-3)
    clocks = clocks_summary(samples)

    # ---- smaller batches (BASELINE.json configs[2]: 1,024 / 4,096 / 16,384 on one stream; 2,048 = a slice of the host pipeline) -------------
    batches = {}
    if rank == 0:
        from lhcb_gen import slice_events
        for nb in (1024, 2048, 4096):
            if nb >= n:
                continue
            sub = DeviceEvents.from_host(slice_events(ev, 0, nb), f"cuda:{local_rank}")
            s2, l2 = ctx.alloc_seeds(nb), ctx.alloc_long(nb)
            w2 = ctx.lhcb_order(sub)
            e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            ts, tm, tc = [], [], []
            for i in range(23):                                      # separately (an event between the kernels)
                e[0].record(stream); ctx.lhcb_order(sub, w2); ctx.lhcb_seeding(sub, s2, workspace=w2); e[1].record(stream)
                ctx.lhcb_matching(s2, sub, l2, workspace=w2); e[2].record(stream); torch.cuda.synchronize()
                if i >= 3:
                    ts.append(e[0].elapsed_time(e[1])); tm.append(e[1].elapsed_time(e[2]))
            for i in range(23):                                      # combined: 10 batches back to back on the stream
                e[0].record(stream)
                for _ in range(10):
                    ctx.lhcb_order(sub, w2); ctx.lhcb_seeding(sub, s2, workspace=w2); ctx.lhcb_matching(s2, sub, l2, workspace=w2)
                e[1].record(stream); torch.cuda.synchronize()
                if i >= 3:
                    tc.append(e[0].elapsed_time(e[1]) / 10)
            comb = nb / np.median(tc) * 1e3
            batches[str(nb)] = {"seeding_events_per_s": nb / np.median(ts) * 1e3, "matching_events_per_s": nb / np.median(tm) * 1e3,
                                "combined_events_per_s": comb, "fraction_of_full_batch_rate": comb / value * world}
            del sub, s2, l2, w2

    # ---- the step before the path, timed on its own: raw unsorted hits -> sorted zones ------
    prepare = None
    if rank == 0:
        from lhcb_gen import shuffle_raw
        raw = shuffle_raw(ev, seed=9)
        up = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dt).view(np.int32 if dt == np.uint32 else dt)).to(f"cuda:{local_rank}")
        ro, rx, rz = up(raw["raw_off"], np.uint32), up(raw["raw_x"], np.float32), up(raw["raw_zone"], np.uint8)
        pout = ctx.lhcb_prepare(ro, rx, rz)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        tp = []
        for i in range(13):
            e[0].record(stream); ctx.lhcb_prepare(ro, rx, rz, pout); e[1].record(stream); torch.cuda.synchronize()
            if i >= 3:
                tp.append(e[0].elapsed_time(e[1]))
        assert int(pout["status"].max().item()) == 0 and torch.equal(pout["hit_x"], dev.hit_x), "lhcb_prepare output differs"
        pb = 13 * rx.numel() + 4 * (ro.numel() + pout["zone_off"].numel())      # x, zone read; x, perm written; offsets
        prepare = {"kernel": "prepare_kernel", "ms": float(np.median(tp)), "events_per_s": n / float(np.median(tp)) * 1e3,
                   "algorithmic_bytes": pb, "achieved_gbs": pb / float(np.median(tp)) / 1e6,
                   "note": "not part of the timed step (BASELINE metric = Seeding+Matching); HBM-bound row, see DESIGN.md"}
        del raw, ro, rx, rz, pout

    # ---- matching with the ghost-killing network, timed on its own ---------------------------
    ghost = None
    if rank == 0:
        from lhcb_gen import ghost_nn
        ctx.lhcb_set_ghost_nn(ghost_nn())
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        tg = []
        for i in range(13):
            e[0].record(stream); ctx.lhcb_matching(seeds, dev, longs, workspace=ws); e[1].record(stream); torch.cuda.synchronize()
            if i >= 3:
                tg.append(e[0].elapsed_time(e[1]))
        n_long_nn = int(longs["count"].sum().item())
        ctx.lhcb_set_ghost_nn(None)
        ctx.lhcb_matching(seeds, dev, longs, workspace=ws); torch.cuda.synchronize()
        ghost = {"matching_ms": float(np.median(tg)), "matching_events_per_s": n / float(np.median(tg)) * 1e3,
                 "long_per_event": n_long_nn / n, "overhead_vs_chi2_ranking": float(np.median(tg)) / float(np.median(match_ms)) - 1.0,
                 "note": "lhcb_matching with lhcb_set_ghost_nn (reading A14b); the timed step uses the chi2 ranking (A14)"}

    # ---- seeding with the Hough-cluster UV version, timed on its own --------------------------
    hough = None
    if rank == 0:
        ctx_h = Context(capacities.with_capacities(ev.geom, capacities.NOMINAL_HOUGH), device=local_rank)
        ctx_h.lhcb_set_uv_hough(True)
        s_h = ctx_h.alloc_seeds(n)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        th_ = []
        for i in range(13):
            e[0].record(stream); ctx_h.lhcb_seeding(dev, s_h); e[1].record(stream); torch.cuda.synchronize()
            if i >= 3:
                th_.append(e[0].elapsed_time(e[1]))
        if int(s_h["status"].max().item()) != 0:
            raise SystemExit("capacity overflow in the Hough-cluster seeding")
        ctx_h.close()
        hough = {"seeding_ms": float(np.median(th_)), "seeding_events_per_s": n / float(np.median(th_)) * 1e3,
                 "seeds_per_event": int(s_h["count"].sum().item()) / n,
                 "note": "lhcb_seeding with lhcb_set_uv_hough (reading A20), capacities.NOMINAL_HOUGH (four CTAs per SM); "
                         "the timed step uses the iterative default"}
        del s_h

    # ---- end to end through the host-buffer C-ABI call ---------------------------------------------------
    e2e = None
    if not args.no_e2e:
        pipe = HostPipeline(ctx, ev, slice_events=2048)
        for _ in range(2):
            pipe.lhcb_reconstruct_host()
        barrier()
        ke = max(3, min(K, 10))
        t = time.perf_counter()
        for _ in range(ke):
            h2d, d2h, launches = pipe.lhcb_reconstruct_host()      # blocks until outputs are on the host
        torch.cuda.synchronize()
        dt = time.perf_counter() - t
        if world > 1:
            tt = torch.tensor([dt], device="cuda"); dist.all_reduce(tt, op=dist.ReduceOp.MAX); dt = float(tt.item())
        n_s_e2e, n_l_e2e = int(pipe._hs.n), int(pipe._hl.n)
        assert n_l_e2e == n_long and n_s_e2e == n_seeds, "end-to-end result differs from the device-resident run"
        bw = pcie_bandwidth(torch, f"cuda:{local_rank}")
        pcie_ms = max(h2d / bw[0], d2h / bw[1]) / 1e6               # each direction alone at its best rate
        replay_ms = pcie_replay(torch, f"cuda:{local_rank}", int(h2d), int(d2h))
        # both directions busy: d2h bytes move at the duplex rates, the rest of the input at the one-way rate
        t_dup = d2h / bw[3] / 1e6
        pcie_duplex_ms = t_dup + max(0.0, h2d - bw[2] * 1e6 * t_dup) / bw[0] / 1e6
        e2e = {"value": world * n * ke / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": 1e3 * dt / ke, "launches_per_step": int(launches),
               "result_bytes": {"seeds": n_s_e2e * 46, "long_tracks": n_l_e2e * 33,
                                "note": "46 B per seed (state, 12 zone-local hit indices, nx, nuv), 33 B per long track, + offsets and status words"},
               "pcie_gbs": {"h2d": bw[0], "d2h": bw[1], "h2d_while_d2h": bw[2], "d2h_while_h2d": bw[3]},
               "pcie_bound_ms": pcie_ms, "fraction_of_pcie_bound": pcie_ms / (1e3 * dt / ke),
               "pcie_duplex_bound_ms": pcie_duplex_ms, "fraction_of_pcie_duplex_bound": pcie_duplex_ms / (1e3 * dt / ke),
               "pcie_replay_ms": replay_ms, "fraction_of_pcie_replay": replay_ms / (1e3 * dt / ke),
               "pcie_note": "pcie_bound: each direction alone at its best rate; pcie_duplex_bound: from the rates measured with both "
                            "directions busy; pcie_replay: the same bytes in the same number of copies, both directions together, "
                            "pinned memory, no kernels (measured in this run): what the box allows for this traffic",
               "api": "lhcb_reconstruct_host (pinned host buffers in, dense seeds + long tracks out; 2048-event slices on three "
                      "streams, one CUDA graph per slice)"}
        pipe.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- CPU baseline (the oracle as it stands) and its step counters: the work model's input ---------------
    cpu = oracle_baseline(ev, args.cpu_sample)
    cnt = cpu["counters_per_event"]

    # ---- roofline of the dominant kernel (seeding_kernel): ALU bound ---------------------------------------
    mean_zone = ev.n_hits / (24.0 * n)
    mean_ut_zone = len(ev.ut_x0) / (4.0 * n)
    ops_seed, ops_match = workmodel.lane_ops(cnt, mean_zone, mean_ut_zone)
    peak = workmodel.alu_peak(1965.0)
    seed_t = float(np.mean(seed_ms)) * 1e-3
    match_t = float(np.mean(match_ms)) * 1e-3
    achieved = ops_seed * n / seed_t
    # seed x VELO pairs inside the |dty| range of Eq. 21, which is all the kernel evaluates (first 1,024 events)
    ne_adm = min(1024, n)
    so = np.concatenate([[0], np.cumsum(np.bincount(sh["event"], minlength=n))])
    adm = 0
    for e_ in range(ne_adm):
        tys = sh["state"][so[e_]:so[e_ + 1], 3]
        tyv = ev.velo_ty[ev.velo_off[e_]:ev.velo_off[e_ + 1]]
        adm += int((np.abs(tys[:, None] - tyv[None, :]) < ev.geom["presel"][3]).sum())
    adm_per_event = adm / ne_adm
    ops_match_adm = adm_per_event * 45 + (ops_match - cnt.get("sv_pairs", 0.0) * 45)
    hbm_bytes = workmodel.hbm_bytes_per_event(ev.n_hits / n, len(ev.velo_x) / n, cnt.get("ut_steps", 0.0), n_seeds / n, n_long / n)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    # ... and the shared-memory bandwidth its searches need (third row): whichever fraction is larger binds
    smem_bytes = 4.0 * workmodel.smem_probe_loads(cnt, mean_zone)
    smem_peak = workmodel.smem_peak(1965.0)
    smem_ach = smem_bytes * n / seed_t
    alu = {"achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "Tlane-op/s", "frac": achieved / peak}
    smem = {"algorithmic_bytes_per_event": smem_bytes, "achieved_tbs": smem_ach / 1e12, "peak_tbs": smem_peak / 1e12,
            "frac": smem_ach / smem_peak, "unit": "TB/s",
            "peak_source": "148 SM x 128 B/clk x 1965 MHz",
            "model": "4-byte probe loads under the binary-search model of workmodel.smem_probe_loads, from the same oracle counters"}
    binds_smem = smem["frac"] > alu["frac"]
    roofline = {"bound": "smem" if binds_smem else "alu", "kernel": "seeding_kernel",
                "achieved": smem["achieved_tbs"] if binds_smem else alu["achieved"],
                "peak": smem["peak_tbs"] if binds_smem else alu["peak"],
                "unit": smem["unit"] if binds_smem else alu["unit"],
                "frac": max(smem["frac"], alu["frac"]), "alu": alu, "smem": smem,
                "traffic": workmodel.NCU_DRAM_BYTES_PER_LAUNCH["seeding_kernel"] if n == 16384 else None,
                "traffic_source": workmodel.NCU_DRAM_SOURCE,
                "counters": "oracle step counters of this run's cpu_baseline leg (%d events)" % cpu["counters_events"],
                "algorithmic_lane_ops_per_event": {"seeding": ops_seed, "matching_all_pairs": ops_match,
                                                   "matching_pairs_in_dty_range": ops_match_adm},
                "kernel_ms": {"seeding": float(np.mean(seed_ms)), "matching": float(np.mean(match_ms))},
                "kernel_share_of_step": {"seeding": float(seed_ms.sum() / (seed_ms.sum() + match_ms.sum())),
                                         "matching": float(match_ms.sum() / (seed_ms.sum() + match_ms.sum()))},
                "matching_frac_all_pairs": ops_match * n / match_t / peak,
                "matching_frac_pairs_in_dty_range": ops_match_adm * n / match_t / peak,
                "matching_note": "all_pairs charges every seed x VELO pair (L279) x 45 lane-ops although the kernel only touches "
                                 "the %.0f of %.0f pairs per event inside the |dty| range of Eq. 21: it measures the method's work, "
                                 "not the kernel's efficiency; pairs_in_dty_range charges only what the kernel evaluates"
                                 % (adm_per_event, cnt.get("sv_pairs", 0.0)),
                "peak_source": "148 SM x 128 lanes x 1965 MHz (B200_PROFILING.md nominal clocks; DESIGN.md)",
                "hbm": {"algorithmic_bytes_per_event": hbm_bytes, "achieved_gbs": hbm_bytes * n / (ms_per_step * 1e-3) / 1e9,
                        "peak_gbs": hbm_peak, "frac": hbm_bytes * n / (ms_per_step * 1e-3) / 1e9 / hbm_peak,
                        "peak_source": "MEASURED_PEAKS.json" if peaks else "fallback B200_PROFILING.md"}}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "cfg3 = BASELINE.json configs[2]: 16,384 nominal-occupancy (mu~5) events, seed 2, "
                                   "one batch of %d events per GPU, lhcb_order + seeding + matching (with UT) on one stream" % n,
                       "events_per_gpu": n, "l2": "inputs (~%.0f MB per batch) exceed the 126 MB L2" % (dev.input_bytes() / 1e6),
                       "parallelism": f"events sharded over {world} GPU(s), no collective",
                       "capacities": "paper_2606_14480_b200.capacities.NOMINAL", "launch": launch},
            "long_tracks_per_s": n_long_all / (ms_per_step * 1e-3), "seeds_per_event": n_seeds / n, "long_per_event": n_long / n,
            "seeding_events_per_s": n / float(np.median(seed_ms)) * 1e3, "matching_events_per_s": n / float(np.median(match_ms)) * 1e3,
            "min_ms": {"seeding": float(seed_ms.min()), "matching": float(match_ms.min())},
            "batches": batches, "prepare": prepare, "ghost_nn": ghost, "uv_hough": hough, "clocks": clocks, "e2e": e2e,
            "gpu_launches": gpu_launches, "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
