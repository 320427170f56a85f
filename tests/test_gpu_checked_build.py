"""-m gpu: the bounds-checked build of the library (nvcc -DGRIDB200_CHECK).  compute-sanitizer is closed on the
measurement pool ("runs under it have left GPUs needing a reset"), so the kernel checks itself: every global address it
forms (atomic flushes, sample gathers, degridding stores) and every shared-memory slot it indexes (raw ring, cooked
arrays, tap table) is tested against its bounds; violations are counted, the access suppressed.  This test runs the
checked library in a subprocess on the shapes that exercise each code path -- several teams per warp, multi-warp teams
(S = 64), tiles (S = 128), padded supports, taps in global memory, both traversals and cell order, ragged tails, off-grid samples,
footprints in the grid's corners -- and requires zero violations AND parity with the oracle.  (Races between the
groups' rings are not covered by this; the ring protocol is two named barriers per batch, grid_warp_kernel.cuh.)"""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r'''
import json, sys
import numpy as np, torch
sys.path.insert(0, sys.argv[1]); sys.path.insert(0, sys.argv[1] + "/tests")
import oracle
from paper_1605_07023_b200 import binding, synth
from gpu_util import errors
oracle.build()
dev = torch.device("cuda:0")
out = []
cases = [(8, 4, 8, 1, None), (16, 1, 8, 32, None), (7, 1, 8, 1, None), (4, 4, 4, 3, None), (64, 2, 2, 2, None),
         (128, 1, 2, 2, None), (32, 4, 8, 300, None), (13, 2, 4, 2, None), (8, 4, 8, 1, dict(pol_split=2))]
for S, P, O, W, extra in cases:
    for mode in (0, 1, 2):                       # channel-innermost, time-innermost, cell order (cell_sort.cuh)
        N = 640 if S >= 64 else 256
        cfg = synth.shrink(synth.get_config("cfg1"), n_ant=8, n_times=37, n_chan=11, grid_size=N)
        rng = np.random.default_rng(S + P)
        uvw = synth.make_uvw(cfg, rng)
        n = uvw.shape[0]
        uvw[:, 2] = rng.uniform(0, W, n)
        e = N // 2 - S // 2 - 1
        uvw[5:25, 0] = np.linspace(e - 2, e + 2, 20); uvw[30:50, 1] = -np.linspace(e - 2, e + 2, 20)   # edges and beyond
        uvw[60:70, :2] = rng.uniform(-0.49 * N, 0.49 * N, (10, 2)); uvw[80, 0] = np.nan
        vis = (rng.standard_normal((n, P)) + 1j * rng.standard_normal((n, P))).astype(np.complex64)
        wts = rng.uniform(0.5, 1, n).astype(np.float32)
        kern = (rng.standard_normal((W, O, S)) + 1j * rng.standard_normal((W, O, S))).astype(np.complex64)
        plan = binding.GridPlan(N, S, O, W, P)
        plan.set_samples(n); plan.set_layout(cfg.n_baselines, cfg.n_times, cfg.n_chan)
        if mode < 2: plan.set_traversal(mode, 16)
        else: plan.set_sample_order(1)
        if extra: plan.set_pol_split(extra["pol_split"])
        plan.set_tuning(batch=8, chunk=40)
        plan.allocate_workspace(dev)
        d = [torch.from_numpy(a).to(dev) for a in (uvw, vis, wts, kern)]
        grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
        plan.execute(*d, grid)
        c1 = plan.debug_counters()
        rel, mx = errors(grid.cpu().numpy(), oracle.grid(N, S, O, W, P, uvw, vis, wts, kern))
        g_in = torch.randn((N, N, P), dtype=torch.complex64, device=dev)
        vo = plan.degrid(d[0], d[2], d[3], g_in)
        c2 = plan.debug_counters()
        ref = oracle.degrid(N, S, O, W, P, uvw, wts, kern, g_in.cpu().numpy())
        drel = float(np.linalg.norm(vo.cpu().numpy() - ref) / np.linalg.norm(ref))
        assert plan.info()["sample_order"] == (1 if mode == 2 else 0)
        out.append(dict(S=S, P=P, W=W, mode=mode, variant=plan.info()["variant"], grid_counters=c1, degrid_counters=c2,
                        rel=float(rel), max_abs=float(mx), degrid_rel=drel))
        plan.destroy()
print("RESULT " + json.dumps(out), flush=True)
import os
os._exit(0)            # skip interpreter teardown (ctypes handles of a second copy of the library)
'''


def test_checked_build_reports_no_violation():
    sys.path.insert(0, ROOT)
    import __graft_entry__ as entry
    lib = entry.build_checked()
    env = dict(os.environ, GRIDB200_LIB=lib)
    r = subprocess.run([sys.executable, "-c", CHILD, ROOT], env=env, capture_output=True, text=True, timeout=1200)
    lines = [l for l in r.stdout.splitlines() if l.startswith("RESULT ")]
    assert r.returncode == 0 and lines, (r.returncode, r.stdout[-1000:], r.stderr[-3000:])
    line = lines[-1]
    res = json.loads(line[len("RESULT "):])
    assert len(res) == 27
    for e in res:
        assert e["variant"] == 3, e
        assert e["grid_counters"] == [0] * 8 and e["degrid_counters"] == [0] * 8, e
        assert e["rel"] <= 1e-5 and e["max_abs"] <= 1e-4 and e["degrid_rel"] <= 1e-5, e
    print(json.dumps(res))
