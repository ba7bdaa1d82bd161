"""lhcb_seeding_static: the Seeding call for code that may not allocate device memory per batch.

Some users of this library sit inside an event loop that was given all its device memory at start-up (the trigger
application the paper's algorithms run in works this way, PAPER.md L35 / L384): a cudaMalloc there would wait
for the whole device to go idle and stall every other stream, and in a process whose memory belongs to another
allocator's pool it would just fail.  For them the library keeps the heaviest-first order tables in a fixed
61,440-byte device array of its own (at most 3,072 events per call) instead of a caller-owned workspace.

What is checked here, on the GPU and through the C-ABI:
  * two calls in a row, on two different batches (the second smaller, so that the first call's leftovers are
    still in the shared array), each give exactly the seeds of the existing path (lhcb_order + lhcb_seeding with a
    torch-owned workspace, and plain lhcb_seeding): same hit sets in the same slot ranges, bit-identical float32
    parameters, same status words -- the tolerance every parity test of this suite uses;
  * the call does not shrink the free device memory (outputs are made beforehand);
  * a batch above the limit is refused with a message that names the limit, and nothing runs.

This file is collected last on purpose (pytest -x stops at the first failure): it must pass alone in a fresh
process and after all other tests.
"""
import ctypes as C
from dataclasses import replace

import numpy as np
import pytest

from lhcb_gen import config, generate

pytestmark = pytest.mark.gpu


def _canonical(ctx, s):
    """Seeds of a batch in a unique order (the order inside a half's slot range is unspecified)."""
    h = ctx.seeds_to_host(s)
    key = np.column_stack([h["event"], h["half"], h["hits"].astype(np.int64)])
    o = np.lexsort(key.T[::-1])
    return dict(key=key[o], state=h["state"][o].view(np.uint32), par=h["par"][o].view(np.uint32), nx=h["nx"][o],
                nuv=h["nuv"][o], status=h["status"], count=s["count"].cpu().numpy())


def _assert_same(a, b, what):
    for name in ("count", "status", "key", "state", "par", "nx", "nuv"):
        assert np.array_equal(a[name], b[name]), (what, name)


def test_static_scratch_seeding_equals_the_workspace_path_on_two_calls_in_a_row():
    from paper_2606_14480_b200 import Context, DeviceEvents, capacities
    torch = pytest.importorskip("torch")
    ev_a = generate(replace(config(2, 300), seed=11))          # nominal occupancy; 600 halves: four waves of CTAs
    ev_b = generate(replace(config(2, 96), seed=12))          # smaller second batch: most of the array keeps call one's words
    ctx = Context(capacities.with_capacities(ev_a.geom))
    try:
        for ev in (ev_a, ev_b):
            dev = DeviceEvents.from_host(ev)
            # the existing path, twice over: with lhcb_order's workspace in torch memory, and without any
            ws = ctx.lhcb_order(dev)
            ref_ws = _canonical(ctx, ctx.lhcb_seeding(dev, workspace=ws))
            ref_plain = _canonical(ctx, ctx.lhcb_seeding(dev))
            _assert_same(ref_ws, ref_plain, "workspace path vs plain path")
            assert len(ref_ws["key"]) > 100 * ev.n_events and not ref_ws["status"].any()
            # the new entry point; outputs exist before the call, poisoned so that stale values cannot pass
            out = ctx.alloc_seeds(dev.n_events)
            for t in out.values():
                if hasattr(t, "fill_"):
                    t.fill_(0x55 if t.dtype == torch.uint8 else 1)
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info(ctx.dev)[0]
            ctx.lhcb_seeding_static(dev, out)
            assert ctx.last_launch_count() == 2           # order + seeding, the library's own kernels
            torch.cuda.synchronize()
            free_after = torch.cuda.mem_get_info(ctx.dev)[0]
            if ev is ev_b:                                # call one may load the module (and with it the array itself)
                assert free_after >= free_before, "the call took device memory"
            _assert_same(ref_ws, _canonical(ctx, out), f"lhcb_seeding_static, {ev.n_events} events")
    finally:
        ctx.close()


def test_static_scratch_seeding_at_exactly_its_limit():
    """3,072 small events (cfg1-like: 40 tracks, no noise) use every word of the built-in array."""
    from paper_2606_14480_b200 import Context, DeviceEvents
    from paper_2606_14480_b200.binding import STATIC_MAX_EVENTS
    ev = generate(config(1, STATIC_MAX_EVENTS))
    ctx = Context(ev.geom)
    try:
        dev = DeviceEvents.from_host(ev)
        ref = _canonical(ctx, ctx.lhcb_seeding(dev))
        assert len(ref["key"]) > 20 * ev.n_events and not ref["status"].any()
        out = ctx.alloc_seeds(dev.n_events)
        _assert_same(ref, _canonical(ctx, ctx.lhcb_seeding_static(dev, out)), "3,072 events")
    finally:
        ctx.close()


def test_static_scratch_seeding_refuses_a_batch_above_its_limit():
    from paper_2606_14480_b200 import Context, DeviceEvents
    from paper_2606_14480_b200.binding import STATIC_MAX_EVENTS, LhcbEvents, LhcbSeeds
    ev = generate(config(1))
    ctx = Context(ev.geom)
    try:
        dev = DeviceEvents.from_host(ev)
        out = ctx.alloc_seeds(dev.n_events)
        out["count"].fill_(7)
        dev.n_events = STATIC_MAX_EVENTS + 1              # the size check comes first: no pointer is followed
        with pytest.raises(RuntimeError, match="3072"):
            ctx.lhcb_seeding_static(dev, out)
        ctx.torch.cuda.synchronize()
        assert (out["count"].cpu().numpy() == 7).all()    # nothing ran
        e, s = LhcbEvents(STATIC_MAX_EVENTS + 1, 0, None, None, None), LhcbSeeds()
        assert ctx.lib.lhcb_seeding_static(ctx._ctx, C.byref(e), C.byref(s), None) == -6
        assert ctx.lib.lhcb_seeding_static(None, C.byref(e), C.byref(s), None) == -4
    finally:
        ctx.close()
