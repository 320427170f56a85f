"""-m gpu: degridding (grid_degrid, the adjoint of grid_execute) through the C ABI against
oracle.degrid, element by element, and the adjoint identity <grid(V), G> = <V, degrid(G)> on the CUDA pair."""
import numpy as np
import pytest

from paper_1605_07023_b200 import synth
from gpu_util import run_gpu

pytestmark = pytest.mark.gpu


def gpu_degrid(N, S, O, W, P, uvw, wts, kernel, grid, layout=None, tuning=None, gather=False):
    import torch
    from paper_1605_07023_b200 import binding
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    try:
        n = uvw.shape[0]
        plan.set_samples(n)
        if layout:
            plan.set_layout(*layout)
        if tuning:
            tuning = dict(tuning)
            if "traversal" in tuning:
                plan.set_traversal(tuning.pop("traversal"), tuning.pop("time_block", 0))
            plan.set_tuning(**tuning)
        if gather:
            plan.set_degrid_gather(1)
        plan.allocate_workspace(dev)
        out = plan.degrid(torch.from_numpy(uvw).to(dev), torch.from_numpy(wts).to(dev),
                          torch.from_numpy(kernel).to(dev), torch.from_numpy(grid.astype(np.complex64)).to(dev))
        torch.cuda.synchronize()
        return out.cpu().numpy()
    finally:
        plan.destroy()


@pytest.mark.parametrize("S,P", [(7, 1), (8, 4), (16, 1), (16, 2), (32, 4), (3, 1), (12, 4), (40, 1)])
def test_degrid_matches_oracle(oracle_mod, S, P):
    # supports below / at / above the lane-group sizes (8, 16, 32), odd and non-power-of-two ones, off-grid
    # and non-finite samples (zeros out), a sample count that is not a multiple of the lane group
    N, O, W, n = 192, 4, 3, 9_973
    uvw, _, wts, kernel = synth.random_problem(90 + S + P, n, N, S, O, W, P, spread=0.52)
    uvw[100:110, 0] = np.nan
    rng = np.random.default_rng(S)
    grid = (rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))).astype(np.complex64)
    ref = oracle_mod.degrid(N, S, O, W, P, uvw, wts, kernel, grid)
    got = gpu_degrid(N, S, O, W, P, uvw, wts, kernel, grid).astype(np.complex128)
    q = oracle_mod.quantise(N, S, O, W, uvw)
    assert (q["valid"] == 0).sum() > 10
    assert not got[q["valid"] == 0].any()                      # skipped samples: exact zeros
    # FP32 sums of S*S terms: error relative to the typical magnitude of an output
    scale = np.sqrt(np.mean(np.abs(ref[q["valid"] == 1]) ** 2))
    assert np.abs(got - ref).max() <= 2e-5 * scale * max(1.0, S / 8)
    assert np.linalg.norm(got - ref) <= 1e-5 * np.linalg.norm(ref)


@pytest.mark.parametrize("S,P,W", [(64, 1, 2), (64, 4, 2), (128, 1, 2), (128, 4, 2), (32, 4, 300), (16, 1, 700), (64, 4, 40), (128, 1, 40)])
def test_degrid_large_supports_and_tables(oracle_mod, S, P, W):
    # degridding with multi-warp teams, tiled bins (S = 128) and tap tables in global memory (many planes)
    N, O, n = 640, 2, 6_007
    uvw, _, wts, kernel = synth.random_problem(300 + S + P + W, n, N, S, O, W, P, spread=0.4, walk=2.0)
    uvw[20:30, 0] = np.nan
    rng = np.random.default_rng(S + W)
    grid = (rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))).astype(np.complex64)
    ref = oracle_mod.degrid(N, S, O, W, P, uvw, wts, kernel, grid)
    got = gpu_degrid(N, S, O, W, P, uvw, wts, kernel, grid).astype(np.complex128)
    via_gather = gpu_degrid(N, S, O, W, P, uvw, wts, kernel, grid, gather=True).astype(np.complex128)
    assert not got[20:30].any()
    assert np.linalg.norm(got - ref) <= 1e-5 * np.linalg.norm(ref)
    assert np.linalg.norm(via_gather - ref) <= 1e-5 * np.linalg.norm(ref)
    assert np.abs(got - ref).max() <= 2e-5 * np.sqrt(np.mean(np.abs(ref) ** 2)) * max(1.0, S / 8)


def test_adjoint_identity_on_gpu(oracle_mod):
    # <grid(V), G> == <V, degrid(G)> with both operators on the GPU (pin P7's identity for the CUDA pair)
    N, S, O, W, P, n = 256, 8, 8, 2, 4, 20_000
    uvw, vis, wts, kernel = synth.random_problem(123, n, N, S, O, W, P, spread=0.45, walk=1.0)
    rng = np.random.default_rng(5)
    G = (rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))).astype(np.complex64)
    gv, _ = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel)
    dg = gpu_degrid(N, S, O, W, P, uvw, wts, kernel, G)
    lhs = np.vdot(gv.astype(np.complex128), G.astype(np.complex128))
    rhs = np.vdot(vis.astype(np.complex128), dg.astype(np.complex128))
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs)


@pytest.mark.parametrize("cu,cv,P,S", [(2, 2, 4, 8), (4, 2, 4, 8), (4, 4, 1, 16), (4, 2, 1, 8), (2, 2, 1, 4),
                                       (8, 4, 1, 32), (4, 4, 2, 16), (2, 2, 2, 8), (8, 4, 1, 16),
                                       (4, 2, 4, 32), (4, 4, 1, 32), (2, 2, 4, 16), (2, 2, 1, 16), (4, 2, 2, 32)])   # teams of 2-8 warps
@pytest.mark.parametrize("mode", [0, 1])
def test_degrid_coarsened_blocks(oracle_mod, cu, cv, P, S, mode):
    # the register-resident kernel (ownership of PAPER.md:63, 77-87 run backwards) for every instantiated
    # block, both traversal orders, small chunks and batches, against the oracle AND the gather kernel
    cfg = synth.shrink(synth.get_config("cfg1"), n_ant=9, n_times=37, n_chan=13, grid_size=384)
    rng = np.random.default_rng(cu * 10 + cv)
    uvw = synth.make_uvw(cfg, rng)
    uvw[50:60, 1] = np.nan
    n = uvw.shape[0]
    N, O, W = cfg.grid_size, 4, 3
    uvw[:, 2] = rng.uniform(0, W, n)
    wts = rng.uniform(0.5, 1.0, n).astype(np.float32)
    kernel = (rng.standard_normal((W, O, S)) + 1j * rng.standard_normal((W, O, S))).astype(np.complex64)
    grid = (rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))).astype(np.complex64)
    ref = oracle_mod.degrid(N, S, O, W, P, uvw, wts, kernel, grid)
    layout = (cfg.n_baselines, cfg.n_times, cfg.n_chan)
    tuning = dict(variant=3, cu=cu, cv=cv, threads_per_cta=1024, batch=16, chunk=64, traversal=mode, time_block=8)
    got = gpu_degrid(N, S, O, W, P, uvw, wts, kernel, grid, layout=layout, tuning=tuning).astype(np.complex128)
    via_gather = gpu_degrid(N, S, O, W, P, uvw, wts, kernel, grid, gather=True).astype(np.complex128)
    assert np.linalg.norm(got - ref) <= 1e-5 * np.linalg.norm(ref)
    assert np.abs(got - ref).max() <= 2e-5 * np.sqrt(np.mean(np.abs(ref) ** 2)) * max(1.0, S / 8)
    assert np.linalg.norm(got - via_gather) <= 2e-5 * np.linalg.norm(ref)
    assert not got[50:60].any()
