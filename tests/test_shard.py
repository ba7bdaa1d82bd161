"""Multi-GPU host logic: events shard across ranks with no data-path collective.
Runs on CPU with the gloo backend, world_size 2 (the kernels themselves are covered by -m gpu)."""
import os
import socket

import numpy as np
import pytest

from lhcb_gen import config, generate, slice_events
from paper_2606_14480_b200 import shard


def test_event_range_partitions_exactly():
    for n in (0, 1, 7, 16, 1000, 16384, 16385):
        for world in (1, 2, 3, 8):
            r = [shard.event_range(k, world, n) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.event_range(2, 2, 10)


def test_weak_chunks_are_disjoint_and_world_independent():
    assert shard.weak_chunks(0, 16384) == (0, 16)
    assert shard.weak_chunks(3, 16384) == (48, 16)
    assert shard.weak_chunks(1, 1500) == (2, 2)
    # a rank's batch is the same events whatever the world size: chunk k is seeded by (seed, k)
    a = generate(config(3, 32), first_chunk=shard.weak_chunks(1, 32)[0])
    b = generate(config(3, 32), first_chunk=1)
    assert np.array_equal(a.hit_x, b.hit_x) and np.array_equal(a.zone_off, b.zone_off)
    c = generate(config(3, 32), first_chunk=0)
    assert not np.array_equal(a.hit_x[:100], c.hit_x[:100])


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, n_events, q):
    import torch.distributed as dist
    from oracle.binding import Oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ev = generate(config(2, n_events))
        a, b = shard.event_range(rank, world, n_events)
        sub = slice_events(ev, a, b)
        s, m = Oracle(ev.geom, "f32").reconstruct(sub)
        ms, tot = shard.reduce_report(10.0 + rank, {"seeds": s["n"], "long": m["n"], "events": b - a})
        q.put((rank, a, b, s["n"], m["n"], ms, tot,
               (s["event"] + a).tolist(), np.asarray(s["hits"]).tolist(), (m["seed"]).tolist()))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_equals_single_process():
    """world_size 2 over gloo: each rank reconstructs its own contiguous event range; the union of
    the shards is the single-process result, and only the report is reduced."""
    import torch.multiprocessing as mp
    from oracle.binding import Oracle
    n, world, port = 6, 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=240) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ev = generate(config(2, n))
    s, m = Oracle(ev.geom, "f32").reconstruct(ev)
    assert [r[1:3] for r in res] == [(0, 3), (3, 6)]
    assert sum(r[3] for r in res) == s["n"] and sum(r[4] for r in res) == m["n"]
    for r in res:                                   # every rank sees the same reduced report
        assert r[5] == 11.0
        assert r[6] == {"seeds": s["n"], "long": m["n"], "events": n}
    # per-event seed hit sets: union of the shards == whole (hit indices are shard-local: rebase them)
    zo = ev.zone_off.astype(np.int64)
    whole = {(int(e),) + tuple(int(x) for x in row) for e, row in zip(s["event"], s["hits"])}
    got = set()
    for r in res:
        base = int(zo[r[1] * 24])
        for e, row in zip(r[7], r[8]):
            got.add((int(e),) + tuple(int(x) + base if x != 0xFFFFFFFF else x for x in row))
    assert got == whole


def test_reduce_report_single_process_is_identity():
    ms, c = shard.reduce_report(3.5, {"a": 2})
    assert ms == 3.5 and c == {"a": 2}
