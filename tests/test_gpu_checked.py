"""The diagnostic build with index checks (-DLHCB_CHECKED) over the whole path.

compute-sanitizer is closed on the GPU pool (profiles/r2_sanitizer.md), so the kernels carry their own checks:
every data-dependent index into a shared-memory queue, table or tile (search results, bin numbers, clone-table
and best-key slots, u/v queues, VELO ranks, UT tile, preparation cells) is compared with its bound; a failure is
recorded, not fatal.  The checked library is a second build of the same sources and must be the only one a process
loads, so the run happens in a child process."""
import json
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

SCRIPT = r"""
import ctypes, json, sys
import numpy as np
from paper_2606_14480_b200.binding import load_library
lib = load_library(checked=True)
lib.lhcb_debug_checks.argtypes = [ctypes.POINTER(ctypes.c_uint * 6), ctypes.c_int]
import torch
from lhcb_gen import config, generate, ghost_nn, shuffle_raw
from paper_2606_14480_b200 import Context, DeviceEvents, capacities

out = {}
buf = (ctypes.c_uint * 6)()
torch.zeros(1, device="cuda")
lib.lhcb_debug_checks(ctypes.byref(buf), 1)
# the checker itself: an index inside its bound passes, one outside (and a negative one) is recorded
lib.lhcb_debug_check_selftest(2, 3); lib.lhcb_debug_check_selftest(5, 3); lib.lhcb_debug_check_selftest(-1, 3)
lib.lhcb_debug_checks(ctypes.byref(buf), 1)
out["selftest"] = dict(failures=int(buf[0]), index=int(buf[2]), bound=int(buf[3]), checks=int(buf[4]))
for name, cfg, n, caps in (("cfg2 defaults", 2, 48, None), ("cfg2 NOMINAL", 2, 48, capacities.NOMINAL),
                           ("cfg4 defaults", 4, 24, None), ("cfg4 NOMINAL_HOUGH", 4, 24, capacities.NOMINAL_HOUGH)):
    ev = generate(config(cfg, n))
    g = dict(ev.geom)
    if caps:
        g.update(caps)
    ctx = Context(g)
    dev = DeviceEvents.from_host(ev)
    ws = ctx.lhcb_order(dev)
    s = ctx.lhcb_seeding(dev, workspace=ws)
    l = ctx.lhcb_matching(s, dev, workspace=ws)
    ctx.lhcb_set_ghost_nn(ghost_nn()); ctx.lhcb_matching(s, dev); ctx.lhcb_set_ghost_nn(None)
    ctx.lhcb_set_uv_hough(True); ctx.lhcb_seeding(dev); ctx.lhcb_set_uv_hough(False)
    raw = shuffle_raw(ev, seed=3)
    up = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dt).view(np.int32 if dt == np.uint32 else dt)).cuda()
    ctx.lhcb_prepare(up(raw["raw_off"], np.uint32), up(raw["raw_x"], np.float32), up(raw["raw_zone"], np.uint8))
    torch.cuda.synchronize()
    lib.lhcb_debug_checks(ctypes.byref(buf), 1)
    out[name] = dict(failures=int(buf[0]), line=int(buf[1]), index=int(buf[2]), bound=int(buf[3]),
                     checks=int(buf[4]) + (int(buf[5]) << 32), seeds=int(s["count"].sum().item()), long=int(l["count"].sum().item()))
    ctx.close()
print("RESULT " + json.dumps(out))
"""


def test_index_checks_find_nothing():
    r = subprocess.run([sys.executable, "-c", SCRIPT], capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [x for x in r.stdout.splitlines() if x.startswith("RESULT ")][-1]
    res = json.loads(line[7:])
    st = res.pop("selftest")
    assert st == dict(failures=2, index=5, bound=3, checks=3), st
    for name, d in res.items():
        assert d["checks"] > 1_000_000, (name, d)            # the checks ran
        assert d["failures"] == 0, (name, d)
        assert d["seeds"] > 0 and d["long"] > 0, (name, d)
