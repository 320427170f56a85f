"""-m gpu: gridding with a dense (non-separable) GCF table (grid_execute_dense) through the C ABI
against oracle.grid_dense."""
import numpy as np
import pytest

from paper_1605_07023_b200 import synth
from gpu_util import assert_parity

pytestmark = pytest.mark.gpu


def gpu_dense(N, S, O, W, P, uvw, vis, wts, k2, layout=None, per_pol=False):
    import torch
    from paper_1605_07023_b200 import binding
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    try:
        n = uvw.shape[0]
        plan.set_samples(n)
        if layout:
            plan.set_layout(*layout)
        plan.allocate_workspace(dev)
        grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
        call = plan.execute_dense_pol if per_pol else plan.execute_dense
        call(torch.from_numpy(uvw).to(dev), torch.from_numpy(np.ascontiguousarray(vis)).to(dev).reshape(n, P),
             torch.from_numpy(wts).to(dev), torch.from_numpy(k2).to(dev), grid)
        torch.cuda.synchronize()
        return grid.cpu().numpy(), plan.last_launches()
    finally:
        plan.destroy()


@pytest.mark.parametrize("S,P,W", [(8, 4, 2), (8, 1, 3), (16, 1, 2), (16, 4, 1), (32, 1, 1), (32, 4, 1), (4, 2, 3), (16, 2, 2),
                                   (7, 1, 2), (12, 4, 1), (40, 1, 1)])
def test_dense_gcf_matches_oracle(oracle_mod, S, P, W):
    # coarsened kernel for power-of-two supports up to 32, one-atomic-per-update kernel otherwise; random
    # non-separable table, off-grid and non-finite samples, ragged sample count
    N, O, n = 200, 3, 12_007
    uvw, vis, wts, _ = synth.random_problem(700 + S + P, n, N, S, O, W, P, spread=0.5, walk=1.2)
    uvw[10:20, 1] = np.nan
    vis[10:20] = np.inf
    rng = np.random.default_rng(S * 7 + P)
    k2 = (rng.standard_normal((W, O, O, S, S)) + 1j * rng.standard_normal((W, O, O, S, S))).astype(np.complex64)
    ref = oracle_mod.grid_dense(N, S, O, W, P, uvw, vis, wts, k2)
    got, launches = gpu_dense(N, S, O, W, P, uvw, vis, wts, k2)
    assert_parity(got, ref, f"dense S={S} P={P} W={W} launches={launches}")


def test_dense_gcf_with_layout_and_separable_limit(oracle_mod):
    # structured samples with the layout hint (time-innermost traversal); a dense table that is an outer product
    # must give the separable path's grid
    cfg = synth.shrink(synth.get_config("cfg1"), n_ant=10, n_times=30, n_chan=12, grid_size=512)
    wl = synth.make_workload(cfg)
    N, S, O, W, P = cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol
    kk = wl.kernel.astype(np.complex128)
    k2 = (kk[:, :, None, :, None] * kk[:, None, :, None, :]).astype(np.complex64)
    ref = oracle_mod.grid_dense(N, S, O, W, P, wl.uvw, wl.vis, wl.weights, k2)
    got, _ = gpu_dense(N, S, O, W, P, wl.uvw, wl.vis, wl.weights, k2, layout=(cfg.n_baselines, cfg.n_times, cfg.n_chan))
    assert_parity(got, ref, "dense with layout")
    sep = oracle_mod.grid(N, S, O, W, P, wl.uvw, wl.vis, wl.weights, wl.kernel)
    assert np.linalg.norm(got - sep) <= 1e-5 * np.linalg.norm(sep)


@pytest.mark.parametrize("S,P,W", [(8, 4, 2), (16, 4, 1), (32, 4, 1), (4, 2, 3), (16, 2, 2), (8, 1, 2), (7, 4, 1), (12, 2, 2), (40, 4, 1)])
def test_dense_gcf_per_polarisation_matches_oracle(oracle_mod, S, P, W):
    # grid_execute_dense_pol (NEXT-4 remainder): an independent random table per polarisation;
    # coarsened kernel for power-of-two supports up to 32, one-atomic-per-update kernel otherwise
    N, O, n = 200, 3, 12_007
    uvw, vis, wts, _ = synth.random_problem(800 + S + P, n, N, S, O, W, P, spread=0.5, walk=1.2)
    uvw[10:20, 1] = np.nan
    vis[10:20] = np.inf
    rng = np.random.default_rng(S * 11 + P)
    k2 = (rng.standard_normal((P, W, O, O, S, S)) + 1j * rng.standard_normal((P, W, O, O, S, S))).astype(np.complex64)
    ref = oracle_mod.grid_dense_pol(N, S, O, W, P, uvw, vis, wts, k2)
    got, launches = gpu_dense(N, S, O, W, P, uvw, vis, wts, k2, per_pol=True)
    assert_parity(got, ref, f"dense per pol S={S} P={P} W={W} launches={launches}")


def test_dense_gcf_per_polarisation_with_layout(oracle_mod):
    # structured samples with the layout hint (time-innermost traversal), 4 different tables
    cfg = synth.shrink(synth.get_config("cfg1"), n_ant=10, n_times=30, n_chan=12, grid_size=512)
    wl = synth.make_workload(cfg)
    N, S, O, W, P = cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol
    rng = np.random.default_rng(77)
    k2 = (rng.standard_normal((P, W, O, O, S, S)) + 1j * rng.standard_normal((P, W, O, O, S, S))).astype(np.complex64)
    ref = oracle_mod.grid_dense_pol(N, S, O, W, P, wl.uvw, wl.vis, wl.weights, k2)
    got, _ = gpu_dense(N, S, O, W, P, wl.uvw, wl.vis, wl.weights, k2, layout=(cfg.n_baselines, cfg.n_times, cfg.n_chan), per_pol=True)
    assert_parity(got, ref, "dense per pol with layout")
