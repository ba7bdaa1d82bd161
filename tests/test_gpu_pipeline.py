"""The end-to-end call lhcb_reconstruct_host (host buffers in, dense host buffers out, CUDA graph per slice)
against the oracle: seeds and long tracks, several slices with a ragged last one."""
import numpy as np
import pytest

from lhcb_gen import config, generate
from oracle.parallel import reconstruct_parallel
from tests.parity import assert_batch_identical

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("nominal", [False, True])
def test_pipeline_output_equals_oracle(nominal):
    from paper_2606_14480_b200 import Context, HostPipeline, capacities
    ev = generate(config(2, 300), workers=4)
    g = dict(ev.geom)
    if nominal:
        g.update(capacities.NOMINAL)
    c = Context(g)
    pipe = HostPipeline(c, ev, slice_events=128, want_par=True)          # slices of 128, 128, 44 events
    for rep in range(2):                                                 # second pass replays the graphs
        h2d, d2h, launches = pipe.lhcb_reconstruct_host()
    gs, gl = pipe.seeds_to_host(), pipe.long_to_host()
    assert not gs["status"].any() and not gl["status"].any()
    os_, om, _ = reconstruct_parallel(ev, workers=4)
    n_s, n_l = assert_batch_identical(os_, om, gs, gl, "pipeline")
    assert n_s > 150 * 300 and n_l > 90 * 300 and launches in (18, 24, 30)
    # offsets: event-half h owns [off[h], off[h+1]) and the long tracks of event e refer to seeds of event e
    assert gs["off"][-1] == n_s and gl["off"][-1] == n_l
    ev_of_seed = np.repeat(np.arange(600), np.diff(gs["off"])) // 2
    assert np.array_equal(ev_of_seed[gl["seed"]], gl["event"])
    # exactly the found entries are copied back: record sizes 74 B per seed (state, hits, par, nx, nuv), 33 B per long track
    want = n_s * (5 * 4 + 12 * 2 + 7 * 4 + 2) + n_l * (4 + 4 + 16 + 1 + 4 + 4) + (600 + 300 + 2 * 3) * 4 + 900 * 4
    assert abs(d2h - want) <= 0.1 * want, (d2h, want)
    # inputs: hits, offsets, VELO states, UT x0 + one row byte per UT hit
    assert h2d < 4 * ev.n_hits + 16 * len(ev.velo_x) + 3 * len(ev.ut_x0) + 300 * 140
    pipe.close()
    c.close()


def test_pipeline_2048_events_last_slice_cut_in_three():
    """One slice of 2,048 events is the whole batch and therefore the last one: it is cut into pieces of 1,024, 512
    and 512 events (the shape of the tail of the batch bench.py times), each with its own graph, order and
    dependent Matching launch.  Seeds and long tracks of all 2,048 events against the oracle."""
    from paper_2606_14480_b200 import Context, HostPipeline, capacities
    ev = generate(config(2, 2048), workers=8)
    c = Context(capacities.with_capacities(ev.geom))
    pipe = HostPipeline(c, ev, slice_events=2048, want_par=True)
    for rep in range(2):
        _, _, launches = pipe.lhcb_reconstruct_host()
    assert launches == 3 * 6                                             # strip decoding, order, seeding, matching, scan, gather
    gs, gl = pipe.seeds_to_host(), pipe.long_to_host()
    assert not gs["status"].any() and not gl["status"].any()
    os_, om, _ = reconstruct_parallel(ev)
    n_s, n_l = assert_batch_identical(os_, om, gs, gl, "pipeline, 2,048 events in 1,024 + 512 + 512")
    assert n_s > 150 * 2048 and n_l > 90 * 2048
    pipe.close()
    c.close()


def test_pipeline_reports_dense_capacity():
    from paper_2606_14480_b200 import Context, HostPipeline
    ev = generate(config(2, 8))
    c = Context(ev.geom)
    pipe = HostPipeline(c, ev, slice_events=4, seeds_per_event=20)
    with pytest.raises(RuntimeError, match="capacit"):
        pipe.lhcb_reconstruct_host()
    pipe.close()
    c.close()


def test_pipeline_cfg3_16384_events_in_the_shape_bench_times(cfg3_full):
    """lhcb_reconstruct_host on the whole cfg3 batch exactly as bench.py's end-to-end leg runs it: NOMINAL
    capacities, slices of 2,048 events (order + seeding + dependent matching + compaction in one graph per slice,
    the last slice cut into 1,024 + 512 + 512), strips shipped as numbers.  Dense seeds and long tracks of all
    16,384 events against the oracle."""
    from paper_2606_14480_b200 import Context, HostPipeline, capacities
    ev, (os_, om, _) = cfg3_full
    c = Context(capacities.with_capacities(ev.geom))
    pipe = HostPipeline(c, ev, slice_events=2048, want_par=True)
    for rep in range(2):
        _, _, launches = pipe.lhcb_reconstruct_host()
    assert launches == 10 * 6                                            # seven full slices + three pieces
    gs, gl = pipe.seeds_to_host(), pipe.long_to_host()
    assert not gs["status"].any() and not gl["status"].any()
    n_s, n_l = assert_batch_identical(os_, om, gs, gl, "pipeline, cfg3 in 2,048-event slices")
    assert n_s > 170 * 16384 and n_l > 100 * 16384
    pipe.close()
    c.close()
