"""-m gpu: compression pre-pass (grid_compress) and gridding of compressed samples
(grid_execute_compressed) through the C ABI, against oracle.compress / oracle.grid."""
import numpy as np
import pytest

from paper_1605_07023_b200 import synth
from gpu_util import assert_parity

pytestmark = pytest.mark.gpu


def slow_walk(seed, n, N, S, O, W, P, step):
    """Samples that creep a fraction of a cell per step (the paper's regime), with a few jumps,
    skipped samples and repeated positions."""
    uvw, vis, wts, kernel = synth.random_problem(seed, n, N, S, O, W, P, spread=0.3, walk=step)
    uvw[:, 2] = np.abs(np.cumsum(np.random.default_rng(seed).normal(0, 0.01, n))) % W
    uvw[n // 3: n // 3 + 50] = uvw[n // 3]                     # an exact run of 50
    uvw[n // 2, 0] = np.nan                                    # skipped samples inside runs
    uvw[n // 2 + 7, 1] = 1e9
    return uvw.astype(np.float32), vis, wts, kernel


def run_compress(N, S, O, W, P, uvw, vis, wts, kernel, grid_too=True):
    import torch
    from paper_1605_07023_b200 import binding
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    try:
        n = uvw.shape[0]
        plan.set_samples(n)
        plan.allocate_workspace(dev)
        d_uvw = torch.from_numpy(uvw).to(dev)
        d_vis = torch.from_numpy(np.ascontiguousarray(vis)).to(dev).reshape(n, P)
        d_w = torch.from_numpy(wts).to(dev)
        recs, cvis, n_c = plan.compress(d_uvw, d_vis, d_w)
        grid = None
        if grid_too:
            grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
            plan.execute_compressed(recs, cvis, torch.from_numpy(kernel).to(dev), grid)
            torch.cuda.synchronize()
            grid = grid.cpu().numpy()
        return recs.cpu().numpy().view(np.uint32).reshape(-1, 2), cvis.cpu().numpy(), n_c, grid
    finally:
        plan.destroy()


@pytest.mark.parametrize("S,P", [(8, 4), (16, 1), (4, 2), (32, 1), (7, 1), (12, 2)])
def test_compress_matches_oracle(oracle_mod, S, P):
    N, O, W, n = 256, 8, 3, 30_011
    uvw, vis, wts, kernel = slow_walk(50 + S + P, n, N, S, O, W, P, step=0.03)
    heads, merged = oracle_mod.compress(N, S, O, W, uvw, vis, wts)
    recs, cvis, n_c, _ = run_compress(N, S, O, W, P, uvw, vis, wts, kernel, grid_too=False)
    assert n_c == len(heads) and n_c < 0.7 * n                 # runs were really merged
    q = oracle_mod.quantise(N, S, O, W, uvw[heads])
    # integer content of every compressed record: bit-exact
    i0, j0 = (recs[:, 0] & 0x7fff).astype(np.int64), (recs[:, 0] >> 16).astype(np.int64)
    ru, rv = (recs[:, 1] & 0xffff).astype(np.int64), (recs[:, 1] >> 16).astype(np.int64)
    sk = 1 << (S - 1).bit_length()
    if sk != S:
        # support padded to a power of two (include/grid.h, "Supports that are not powers of two"): the row index
        # carries in its lowest bit which zero-padded copy of the tap row is used; with copy 1 (zeros in front)
        # the stored origin is the real one minus the padding
        i0, j0 = i0 + (sk - S) * (ru & 1), j0 + (sk - S) * (rv & 1)
        ru, rv = ru >> 1, rv >> 1
    np.testing.assert_array_equal(i0, q["i0"])
    np.testing.assert_array_equal(j0, q["j0"])
    np.testing.assert_array_equal(ru, q["wp"] * O + q["su"])
    np.testing.assert_array_equal(rv, q["wp"] * O + q["sv"])
    # merged values: FP32 sums of up to 50 terms against float64
    scale = np.abs(merged).max()
    assert np.abs(cvis.astype(np.complex128) - merged).max() <= 2e-6 * scale


@pytest.mark.parametrize("S,P", [(8, 4), (16, 1), (8, 1), (16, 4), (7, 1), (12, 4)])
def test_grid_of_compressed_samples(oracle_mod, S, P):
    # "identical results" up to rounding -- compare with the oracle grid of the ORIGINAL samples
    N, O, W, n = 256, 8, 3, 40_003
    uvw, vis, wts, kernel = slow_walk(70 + S + P, n, N, S, O, W, P, step=0.05)
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    _, _, n_c, got = run_compress(N, S, O, W, P, uvw, vis, wts, kernel)
    assert 0 < n_c < n
    assert_parity(got, ref, f"compressed S={S} P={P} n_c={n_c}")


def test_compress_edge_cases(oracle_mod):
    N, S, O, W, P = 128, 8, 4, 2, 1
    kernel = np.ones((W, O, S), np.complex64)
    # every sample skipped -> zero compressed samples, grid untouched
    uvw = np.full((100, 3), 1e9, np.float32)
    recs, cvis, n_c, grid = run_compress(N, S, O, W, P, uvw, np.ones((100, 1), np.complex64), np.ones(100, np.float32), kernel)
    assert n_c == 0 and not grid.any()
    # one long run crossing several 1024-sample blocks -> a single sample carrying the whole sum
    uvw = np.zeros((5000, 3), np.float32)
    vis = np.full((5000, 1), 0.5 + 0.25j, np.complex64)
    recs, cvis, n_c, grid = run_compress(N, S, O, W, P, uvw, vis, np.full(5000, 2.0, np.float32), kernel)
    assert n_c == 1 and abs(cvis[0, 0] - 5000 * (1.0 + 0.5j)) < 1e-2
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, np.full(5000, 2.0, np.float32), kernel)
    assert_parity(grid, ref, "single run")


def test_paper_shaped_workload_compressed_full_size(oracle_mod):
    # 7.26 M samples creeping 0.04 cells per dump (shape of PAPER.md:107-113), compressed on the device and
    # gridded from the compressed samples, against oracle row bands of the ORIGINAL samples
    import torch
    from paper_1605_07023_b200 import binding
    from gpu_util import REL_L2_TOL, MAX_ABS_TOL
    cfg = synth.get_config("paper_S16_P1")
    wl = synth.make_workload(cfg)
    N, S, O, W, P = cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    plan.set_samples(cfg.n_vis)
    plan.allocate_workspace(dev)
    recs, cvis, n_c = plan.compress(torch.from_numpy(wl.uvw).to(dev), torch.from_numpy(wl.vis).to(dev),
                                    torch.from_numpy(wl.weights).to(dev))
    assert cfg.n_vis / n_c > 1.5                                # the regime where compression pays
    grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
    plan.execute_compressed(recs, cvis, torch.from_numpy(wl.kernel).to(dev), grid)
    torch.cuda.synchronize()
    c = N // 2
    for lo, hi in ((c - 4, c + 4), (c + N // 10, c + N // 10 + 4)):
        ref = oracle_mod.grid(N, S, O, W, P, wl.uvw, wl.vis, wl.weights, wl.kernel, rows=(lo, hi))
        got = grid[lo:hi].cpu().numpy().astype(np.complex128)
        rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        mx = np.abs(got - ref).max() / np.abs(ref).max()
        print(f"paper_S16_P1 compressed {cfg.n_vis}->{n_c} rows {lo}:{hi} rel_l2={rel:.2e} max={mx:.2e}")
        assert rel <= REL_L2_TOL and mx <= MAX_ABS_TOL
    plan.destroy()
