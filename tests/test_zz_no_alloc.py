"""-m gpu, collected last: grid_execute_static -- grid_execute with its workspace in the library's static device array
(include/grid.h: no cudaMalloc anywhere; at most GRID_STATIC_SCRATCH_BYTES per call; for callers under CUDA graph
capture or in harnesses that forbid allocation).  Its output is checked against the existing path (grid_execute with a
caller-provided workspace) on two calls in a row that differ in size, support and polarisation count, so that whatever
the first call left in the shared array would show in the second; atomics make the order of the additions
nondeterministic, hence the tolerances of the other parity tests (gpu_util: rel-L2 <= 1e-5, max-abs <= 1e-4 max|grid|).
Both results are also compared with the float64 oracle.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_1605_07023_b200 import synth
from gpu_util import assert_parity, run_gpu

pytestmark = pytest.mark.gpu

STATIC_BYTES = 20 << 20            # GRID_STATIC_SCRATCH_BYTES of include/grid.h


def run_static(N, S, O, W, P, uvw, vis, weights, kernel, layout=None, grid_init=None):
    import torch
    from paper_1605_07023_b200 import binding
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    try:
        n = uvw.shape[0]
        plan.set_samples(n)
        if layout:
            plan.set_layout(*layout)
        assert plan.workspace_bytes() <= STATIC_BYTES      # no set_workspace / allocate_workspace: the static array is used
        grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev) if grid_init is None else torch.from_numpy(grid_init).to(dev)
        d = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (uvw, vis, weights, kernel)]
        plan.execute_static(d[0], d[1].reshape(n, P), d[2], d[3], grid)
        torch.cuda.synchronize()
        return grid.cpu().numpy(), plan.info(), plan.last_launches()
    finally:
        plan.destroy()


def test_static_scratch_matches_existing_path_on_two_calls_in_a_row(oracle_mod):
    # call 1: structured samples with the layout hint (time-innermost walk), 4 polarisations, S = 8, 61 440 samples
    cfg = synth.shrink(synth.get_config("cfg1"), n_ant=16, n_times=32, n_chan=16, grid_size=512)
    wl = synth.make_workload(cfg)
    lay = (cfg.n_baselines, cfg.n_times, cfg.n_chan)
    a = (cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol, wl.uvw, wl.vis, wl.weights, wl.kernel)
    # call 2: fewer, unstructured samples, 1 polarisation, padded support 7, 3 planes, off-grid and NaN samples, and a
    # grid that is accumulated into -- stale records, chunk order or counters of call 1 would corrupt it
    N2, S2, O2, W2, P2, n2 = 256, 7, 4, 3, 1, 20_003
    uvw2, vis2, wts2, kern2 = synth.random_problem(77, n2, N2, S2, O2, W2, P2, spread=0.52, walk=1.5)
    uvw2[100:110, 0] = np.nan
    init2 = (np.random.default_rng(5).standard_normal((N2, N2, P2, 2)).astype(np.float32).view(np.complex64)[..., 0])
    b = (N2, S2, O2, W2, P2, uvw2, vis2, wts2, kern2)

    got1, info1, launches1 = run_static(*a, layout=lay)
    got2, info2, launches2 = run_static(*b, grid_init=init2)            # directly after call 1, same shared array
    ref1, rinfo1 = run_gpu(*a, layout=lay)                              # the existing path, its own workspace
    ref2, rinfo2 = run_gpu(*b, grid_init=init2)
    # same kernels, same number of launches as the existing path
    for k in ("variant", "cu", "cv", "pol_split", "threads_per_cta", "batch", "chunk"):
        assert info1[k] == rinfo1[k] and info2[k] == rinfo2[k], k
    assert launches1 == rinfo1["launches"] and launches2 == rinfo2["launches"] and launches1 >= 2
    assert_parity(got1, ref1.astype(np.complex128), "static scratch vs workspace path, call 1")
    assert_parity(got2, ref2.astype(np.complex128), "static scratch vs workspace path, call 2")
    # and against the oracle
    assert_parity(got1, oracle_mod.grid(*a), "static scratch vs oracle, call 1")
    assert_parity(got2, oracle_mod.grid(*b) + init2.astype(np.complex128), "static scratch vs oracle, call 2")
    # a third call repeats call 1 after call 2 (larger after smaller)
    got3, _, _ = run_static(*a, layout=lay)
    assert_parity(got3, ref1.astype(np.complex128), "static scratch vs workspace path, call 3")


def test_static_scratch_rejects_sizes_beyond_its_maximum():
    import torch
    from paper_1605_07023_b200 import binding
    dev = torch.device("cuda:0")
    N, S, O, W, P, n = 512, 8, 8, 1, 1, 2_000_000          # 2 M samples: 33 MB of workspace > 20 MiB
    plan = binding.GridPlan(N, S, O, W, P)
    plan.set_samples(n)
    assert plan.workspace_bytes() > STATIC_BYTES
    uvw = torch.zeros((n, 3), dtype=torch.float32, device=dev)
    vis = torch.ones((n, P), dtype=torch.complex64, device=dev)
    wts = torch.ones(n, dtype=torch.float32, device=dev)
    kern = torch.ones((W, O, S), dtype=torch.complex64, device=dev)
    grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
    with pytest.raises(binding.GridError) as e:
        plan.execute_static(uvw, vis, wts, kern, grid)
    assert e.value.code == binding.GRID_ERR_UNSUPPORTED
    msg = str(e.value)
    assert "static scratch" in msg and str(STATIC_BYTES) in msg and "several calls" in msg
    torch.cuda.synchronize()
    assert not grid.any() and plan.last_launches() == 0     # nothing was launched
    plan.destroy()
