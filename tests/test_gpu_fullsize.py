"""-m gpu: BASELINE.json's configs at FULL size, in the launch configuration bench.py times (plan
defaults + layout hint), against the float64 oracle on what it can compute in seconds:
  * sampled outputs: bands of grid rows (centre, mid-radius, outer) computed exactly by the oracle
    (its row-restricted mode scans every sample), compared element by element with the north_star
    tolerances, the max-abs one relative to the band's own maximum (stricter than max|grid|);
  * a property that holds at any size (pin P3): with V = 1 the sum of the grid equals
    sum_n weight_n * ksum[wp][sv] * ksum[wp][su]; a lost or doubled chunk of 1024 samples moves it by
    3e-5, the bound is 1e-5 of the sum of the terms' moduli;
  * step a1 bit-exact on a strided sample of the full uvw array.
"""
import numpy as np
import pytest

from paper_1605_07023_b200 import synth
from gpu_util import REL_L2_TOL, MAX_ABS_TOL

pytestmark = pytest.mark.gpu

# every BASELINE.json config and all eight points of the config-4 sweep, each with the plan's default tuning
FULL = ["cfg1", "cfg2", "cfg3", "cfg4_S4_P1", "cfg4_S4_P4", "cfg4_S8_P1", "cfg4_S8_P4", "cfg4_S16_P1", "cfg4_S16_P4",
        "cfg4_S32_P1", "cfg4_S32_P4"]


def _bands(N, S):
    c = N // 2
    return [(c - 8, c + 8), (c + N // 8, c + N // 8 + 8), (c - int(0.4 * N), c - int(0.4 * N) + 8)]


@pytest.mark.parametrize("name", FULL)
def test_full_size(oracle_mod, name):
    import torch
    from paper_1605_07023_b200 import binding
    cfg = synth.get_config(name)
    wl = synth.make_workload(cfg)
    N, S, O, W, P = cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol
    dev = torch.device("cuda:0")
    d_uvw, d_vis, d_w, d_k = (torch.from_numpy(a).to(dev) for a in (wl.uvw, wl.vis, wl.weights, wl.kernel))
    plan = binding.GridPlan(N, S, O, W, P)
    plan.set_samples(cfg.n_vis)
    plan.set_layout(cfg.n_baselines, cfg.n_times, cfg.n_chan)
    plan.allocate_workspace(dev)
    grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
    plan.execute(d_uvw, d_vis, d_w, d_k, grid)
    torch.cuda.synchronize()

    # a1 on a strided sample of the full array: bit-exact
    step = 997
    q_gpu = plan.quantise(d_uvw[::step].contiguous()).cpu().numpy()
    q_ref = oracle_mod.quantise(N, S, O, W, wl.uvw[::step])
    for col, key in enumerate(("i0", "j0", "su", "sv", "wp", "valid")):
        assert np.array_equal(q_gpu[:, col], q_ref[key].astype(np.int32)), key

    # sampled outputs: exact row bands
    for lo, hi in _bands(N, S):
        ref = oracle_mod.grid(N, S, O, W, P, wl.uvw, wl.vis, wl.weights, wl.kernel, rows=(lo, hi))
        got = grid[lo:hi].cpu().numpy().astype(np.complex128)
        nref = np.linalg.norm(ref.ravel())
        assert nref > 0, f"{name}: empty band {lo}:{hi}"
        rel = np.linalg.norm((got - ref).ravel()) / nref
        mx = np.abs(got - ref).max() / np.abs(ref).max()
        print(f"{name} rows {lo}:{hi} rel_l2={rel:.2e} max_abs/max={mx:.2e}")
        assert rel <= REL_L2_TOL and mx <= MAX_ABS_TOL, (name, lo, hi, rel, mx)

    # property at full size: V = 1  =>  sum(grid) = sum_n w_n * ksum_v * ksum_u
    ones = torch.ones_like(d_vis)
    grid.zero_()
    plan.execute(d_uvw, ones, d_w, d_k, grid)
    torch.cuda.synchronize()
    total = grid.to(torch.complex128).sum(dim=(0, 1)).cpu().numpy()
    q = oracle_mod.quantise(N, S, O, W, wl.uvw)
    ok = q["valid"] == 1
    ksum = wl.kernel.astype(np.complex128).sum(axis=2)                 # [W][O]
    terms = wl.weights[ok].astype(np.float64) * ksum[q["wp"][ok], q["sv"][ok]] * ksum[q["wp"][ok], q["su"][ok]]
    expect, scale = terms.sum(), np.abs(terms).sum()
    err = np.abs(total - expect).max() / scale
    print(f"{name} sum property: err/scale={err:.2e} n_valid={int(ok.sum())}")
    assert err <= 1e-5, (name, err)
    plan.destroy()


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3"])
def test_full_size_degrid_sampled(oracle_mod, name):
    # grid_degrid at full size in the configuration bench.py --op degrid times: the oracle computes a strided
    # sample of the outputs one by one (each needs only its own footprint of the same random grid)
    import torch
    from paper_1605_07023_b200 import binding
    cfg = synth.get_config(name)
    rng = np.random.default_rng(cfg.seed)
    uvw = synth.make_uvw(cfg, rng)
    N, S, O, W, P = cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol
    kernel = synth.make_kernel(cfg, rng)
    wts = np.random.default_rng(1).uniform(0.5, 1.0, cfg.n_vis).astype(np.float32)
    dev = torch.device("cuda:0")
    torch.manual_seed(7)
    d_grid = torch.randn((N, N, P), dtype=torch.complex64, device=dev)
    plan = binding.GridPlan(N, S, O, W, P)
    plan.set_samples(cfg.n_vis)
    plan.set_layout(cfg.n_baselines, cfg.n_times, cfg.n_chan)
    plan.allocate_workspace(dev)
    out = plan.degrid(torch.from_numpy(uvw).to(dev), torch.from_numpy(wts).to(dev), torch.from_numpy(kernel).to(dev), d_grid)
    torch.cuda.synchronize()
    step = 4999
    got = out[::step].cpu().numpy().astype(np.complex128)
    ref = oracle_mod.degrid(N, S, O, W, P, uvw[::step], wts[::step], kernel, d_grid.cpu().numpy())
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    print(f"{name} degrid sampled ({len(ref)} outputs): rel_l2={rel:.2e}")
    assert rel <= REL_L2_TOL
    assert np.abs(got - ref).max() <= 2e-5 * np.sqrt(np.mean(np.abs(ref) ** 2)) * max(1.0, S / 8)
    # every output was written: no sample left at the allocation's garbage (finite everywhere, right count of zeros)
    assert bool(torch.isfinite(torch.view_as_real(out)).all())
    plan.destroy()


@pytest.mark.parametrize("N,P,S", [(32767, 1, 8), (16001, 4, 16)])
def test_maximum_grid_size_corners(oracle_mod, N, P, S):
    # the largest grid the ABI accepts (N = 32767, odd: rows are not 16-byte aligned) and an odd 4-pol one
    # beyond 2^31 bytes: samples in the four corners, on the last valid cell, and in the centre -- 32/64-bit
    # index arithmetic of the flush addresses.  The oracle computes the touched row bands only.
    import torch
    from paper_1605_07023_b200 import binding
    O, W = 4, 2
    rng = np.random.default_rng(N)
    half = N // 2
    lo_u, hi_u = -half + S / 2.0, N - 1 - half - S / 2.0 + 0.4          # first / last footprint that still fits
    corners = [(lo_u, lo_u), (lo_u, hi_u), (hi_u, lo_u), (hi_u, hi_u), (0.3, -0.2), (hi_u + 1.0, 0.0)]   # last one: off grid
    uv = np.repeat(np.array(corners, dtype=np.float64), 40, axis=0) + rng.uniform(-0.4, 0.0, (40 * len(corners), 2))
    n = len(uv)
    uvw = np.concatenate([uv, rng.uniform(0, W, (n, 1))], axis=1).astype(np.float32)
    vis = (rng.standard_normal((n, P)) + 1j * rng.standard_normal((n, P))).astype(np.complex64)
    wts = rng.uniform(0.5, 1, n).astype(np.float32)
    kernel = (rng.standard_normal((W, O, S)) + 1j * rng.standard_normal((W, O, S))).astype(np.complex64)
    q = oracle_mod.quantise(N, S, O, W, uvw)
    assert q["valid"][:200].all() and not q["valid"][200:].any()
    assert q["i0"][:200].min() == 0 and (q["i0"][:200] + S).max() == N and (q["j0"][:200] + S).max() == N
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    plan.set_samples(n)
    plan.allocate_workspace(dev)
    grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
    plan.execute(torch.from_numpy(uvw).to(dev), torch.from_numpy(vis).to(dev), torch.from_numpy(wts).to(dev),
                 torch.from_numpy(kernel).to(dev), grid)
    torch.cuda.synchronize()
    touched = 0
    for lo, hi in ((0, 2 * S), (half - 2 * S, half + 2 * S), (N - 2 * S, N)):
        ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel, rows=(lo, hi))
        got = grid[lo:hi].cpu().numpy().astype(np.complex128)
        assert np.abs(ref).max() > 0
        assert np.linalg.norm(got - ref) <= REL_L2_TOL * np.linalg.norm(ref)
        assert np.abs(got - ref).max() <= MAX_ABS_TOL * np.abs(ref).max()
        touched += int((got != 0).sum())
    # nothing landed anywhere else
    assert int((torch.view_as_real(grid) != 0).any(dim=-1).sum().item()) == touched
    plan.destroy()
