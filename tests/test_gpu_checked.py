"""The CHECKED build of the library (libimager_checked.so, -DIMAGER_CHECKED=1, include/imager.h imager_debug_violations):
every index the planner and the tiled kernels form is tested against its bounds on the device.  compute-sanitizer is
closed on this GPU pool, so this is the memory-safety evidence of the hand-managed parts: hit-record
places, visibility indices of hits, shared-memory tap addresses, strips, item and block ranges, the duplicate hash table,
the planner's strip windows.  Workloads: config 1, config 2 in full and with every 20th time step (block splitting, the two-ended
queue, multi-group units), a cut of config 3 (4 x 4 Mueller elements), config 4's even support 64, dropped and invalid
input, duplicates.  Runs in a subprocess because a process loads one libimager."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import json, sys
import numpy as np, torch
sys.path.insert(0, %(root)r)
from paper_2206_15117_b200 import Plan, load_library
from paper_2206_15117_b200.binding import c_int64
from synth import make_workload

def run(wl, corrupt=False):
    p = wl.params
    n, npol, nc = p["grid_size"], p["n_pol"], p["n_corr"]
    uvw_h = wl.uvw.copy()
    if corrupt:                       # invalid and far-out input: dropped (R8, R17), never indexed
        uvw_h[::7, 0] = np.nan
        uvw_h[3::11, 1] *= 50.0
        uvw_h[5::13] = uvw_h[4::13][: len(uvw_h[5::13])]      # exact duplicates
    with Plan(p, wl.nvis) as plan:
        uvw = torch.from_numpy(uvw_h).cuda()
        vis = torch.from_numpy(wl.vis).cuda()
        wts = torch.from_numpy(wl.weights).cuda()
        a = torch.from_numpy(wl.a_index).cuda() if wl.a_index is not None else None
        grid = torch.zeros((npol, n, n), dtype=torch.complex64, device="cuda")
        out = torch.zeros((wl.nvis, nc), dtype=torch.complex64, device="cuda")
        plan.grid(uvw, vis, wts, grid, a)
        plan.degrid(uvw, grid, out, a, flags=1)
        plan.degrid(uvw, grid, out, a)                        # re-index, residual flag off
        torch.cuda.synchronize()
        assert torch.isfinite(torch.view_as_real(grid)).all() and torch.isfinite(torch.view_as_real(out)).all()
        return plan.index_stats()["n_hits"]

hits = {}
hits["config1"] = run(make_workload("config1"))
hits["config2"] = run(make_workload("config2"))
hits["config2/20"] = run(make_workload("config2", time_stride=20))
hits["config2/20 corrupt"] = run(make_workload("config2", time_stride=20), corrupt=True)
hits["config3/100"] = run(make_workload("config3", time_stride=100))
hits["config4/10"] = run(make_workload("config4", time_stride=10))
v = (c_int64 * 16)()
rc = load_library().imager_debug_violations(v)
print("RESULT " + json.dumps({"checked": rc, "violations": list(v), "hits": hits}))
"""


def test_checked_build_reports_no_violation():
    import torch
    assert torch.cuda.is_available()
    from paper_2206_15117_b200 import build as lib_build
    lib = lib_build.build(checked=True)
    env = dict(os.environ, IMAGER_LIBRARY=lib)
    r = subprocess.run([sys.executable, "-c", SCRIPT % {"root": ROOT}], env=env, capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, r.stderr[-3000:]
    res = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("RESULT ")][-1][7:])
    assert res["checked"] == 1, "IMAGER_LIBRARY did not select the checked build"
    assert all(h > 0 for h in res["hits"].values()), res
    assert res["violations"] == [0] * 16, res


def test_normal_build_says_it_is_unchecked():
    from paper_2206_15117_b200 import load_library
    from paper_2206_15117_b200.binding import c_int64
    v = (c_int64 * 16)()
    rc = load_library().imager_debug_violations(v)
    if os.environ.get("IMAGER_LIBRARY"):
        pytest.skip("an alternative library is selected")
    assert rc == 0 and list(v) == [0] * 16
