"""-m gpu: grid_execute with the samples sorted by grid cell in the a1 pass (grid_plan_set_sample_order,
csrc/cell_sort.cuh) against the float64 oracle on the same seeded inputs, through the C ABI.  The sum is
order-independent (pin P11), so the tolerances are the ones of every other gridding test (R20)."""
import numpy as np
import pytest

from paper_1605_07023_b200 import synth
from gpu_util import assert_parity, run_gpu

pytestmark = pytest.mark.gpu

# every instantiated block of the warp kernel
WARP = [(2, 2, 1), (4, 2, 1), (4, 4, 1), (8, 4, 1), (2, 2, 2), (4, 2, 2), (4, 4, 2), (2, 2, 4), (4, 2, 4)]


@pytest.mark.parametrize("cu,cv,P", WARP)
@pytest.mark.parametrize("S", [4, 8, 16, 32])
def test_cell_order_every_warp_block(oracle_mod, cu, cv, P, S):
    # ragged tail (n not a multiple of 4, batch or chunk), samples off the grid and with non-finite coordinates
    # (they sort behind all others and must contribute exact zeros), jumps larger than the support, 3 planes
    if cu > S or cv > S:
        pytest.skip("block larger than the support")
    N, O, W, n = 128, 4, 3, 20_003
    uvw, vis, wts, kernel = synth.random_problem(7000 + 100 * cu + 10 * cv + P + S, n, N, S, O, W, P,
                                                 spread=0.5, walk=1.5)
    uvw[7000:7010, 0] = np.nan
    vis[7000:7010] = np.inf
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    for batch, chunk in ((32, 300), (8, 64)):
        got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel,
                            tuning=dict(sample_order=1, variant=3, cu=cu, cv=cv, threads_per_cta=1024, batch=batch, chunk=chunk))
        assert (info["variant"], info["cu"], info["cv"], info["sample_order"]) == (3, cu, cv, 1)
        assert info["launches"] == 6, info                       # count, three scan kernels, scatter, gridding
        assert_parity(got, ref, f"cell order C={cu}x{cv} P={P} S={S} batch={batch} {info}")


@pytest.mark.parametrize("cu,cv", [(2, 2), (4, 2), (4, 4)])
@pytest.mark.parametrize("S", [8, 16])
def test_cell_order_pol_split(oracle_mod, cu, cv, S):
    N, O, W, P, n = 160, 8, 2, 4, 15_001
    uvw, vis, wts, kernel = synth.random_problem(7500 + 10 * cu + cv + S, n, N, S, O, W, P, spread=0.45, walk=0.8)
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel,
                        tuning=dict(sample_order=1, variant=3, cu=cu, cv=cv, pol_split=2))
    assert (info["pol_split"], info["sample_order"]) == (2, 1)
    assert_parity(got, ref, f"cell order C={cu}x{cv} PS=2 S={S}")


@pytest.mark.parametrize("S,P,N", [(7, 1, 512), (12, 4, 200), (13, 2, 97), (3, 1, 64), (40, 1, 300), (64, 4, 256),
                                   (100, 1, 512), (128, 1, 512)])
def test_cell_order_padded_and_large_supports(oracle_mod, S, P, N):
    # supports that are not powers of two (zero-padded taps: the key is the cell of the PADDED footprint's origin),
    # 64-bit masks (S = 64) and tiled bins (S = 128: four queue entries per chunk)
    O, W, n = 4, 2, 6_007
    uvw, vis, wts, kernel = synth.random_problem(7700 + S + P, n, N, S, O, W, P, spread=0.5, walk=2.0)
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, tuning=dict(sample_order=1))
    assert (info["variant"], info["sample_order"]) == (3, 1), info
    assert_parity(got, ref, f"cell order S={S} P={P} N={N} {info}")


def test_cell_order_degenerate_inputs(oracle_mod):
    N, S, O, W, P = 64, 8, 8, 1, 4
    rng = np.random.default_rng(5)
    kernel = (rng.normal(size=(W, O, S)) + 1j * rng.normal(size=(W, O, S))).astype(np.complex64)
    # (a) every sample in ONE cell (one histogram bin takes all the atomics; every chunk flushes once)
    n = 50_001
    uvw = np.zeros((n, 3), np.float32)
    uvw[:, :2] = rng.uniform(0.0, 0.99, (n, 2)) + 3.0
    vis = (rng.normal(size=(n, P)) + 1j * rng.normal(size=(n, P))).astype(np.complex64)
    wts = rng.uniform(0.5, 1.0, n).astype(np.float32)
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, _ = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, tuning=dict(sample_order=1))
    assert_parity(got, ref, "one cell")
    # (b) every sample off the grid: the grid must stay exactly as it was
    uvw_off = uvw + 1000.0
    init = (rng.normal(size=(N, N, P)) + 1j * rng.normal(size=(N, N, P))).astype(np.complex64)
    got, _ = run_gpu(N, S, O, W, P, uvw_off, vis, wts, kernel, tuning=dict(sample_order=1), grid_init=init)
    assert np.array_equal(got, init)
    # (c) one sample; (d) grid accumulated into (R10)
    got, _ = run_gpu(N, S, O, W, P, uvw[:1], vis[:1], wts[:1], kernel, tuning=dict(sample_order=1), grid_init=init)
    ref1 = oracle_mod.grid(N, S, O, W, P, uvw[:1], vis[:1], wts[:1], kernel) + init
    assert_parity(got, ref1, "one sample onto a non-zero grid")


def test_cell_order_edges_and_corners(oracle_mod):
    # odd grid size whose N*N + 1 histogram entries are not a multiple of the scan tile, footprints in all four
    # corners (first and last histogram bins), one polarisation (records carry the pre-weighted visibility)
    N, S, O, W, P = 1001, 8, 8, 1, 1
    rng = np.random.default_rng(11)
    n = 40_003
    uvw = np.zeros((n, 3), np.float32)
    lo, hi = -(N // 2) + S / 2 - 1, (N - 1 - N // 2) - S / 2
    uvw[:, 0] = rng.choice([lo + 0.3, hi + 0.4, 0.0], n) + rng.uniform(-0.2, 0.2, n)
    uvw[:, 1] = rng.choice([lo + 0.3, hi + 0.4, 0.0], n) + rng.uniform(-0.2, 0.2, n)
    vis = (rng.normal(size=(n, P)) + 1j * rng.normal(size=(n, P))).astype(np.complex64)
    wts = rng.uniform(0.5, 1.0, n).astype(np.float32)
    kernel = (rng.normal(size=(W, O, S)) + 1j * rng.normal(size=(W, O, S))).astype(np.complex64)
    q = oracle_mod.quantise(N, S, O, W, uvw)
    assert q["valid"].all() and q["i0"].min() == 0 and q["j0"].min() == 0 and q["i0"].max() == N - S and q["j0"].max() == N - S
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, tuning=dict(sample_order=1))
    assert info["sample_order"] == 1
    assert_parity(got, ref, "corners")


def test_cell_order_is_the_default_for_large_inputs(oracle_mod):
    # automatic mode: 2^20 samples or more on a grid of at most 8 n_vis cells; same answer as input order
    cfg = synth.shrink(synth.get_config("cfg1"), n_ant=24, n_times=64, n_chan=64, grid_size=1024)
    wl = synth.make_workload(cfg)
    assert cfg.n_vis >= 1 << 20
    args = (cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol, wl.uvw, wl.vis, wl.weights, wl.kernel)
    layout = (cfg.n_baselines, cfg.n_times, cfg.n_chan)
    got, info = run_gpu(*args, layout=layout)
    assert info["sample_order"] == 1 and info["launches"] == 6, info
    got0, info0 = run_gpu(*args, layout=layout, tuning=dict(sample_order=0))
    assert info0["sample_order"] == 0 and info0["launches"] == 2, info0
    lo = cfg.grid_size // 2 + 40
    ref = oracle_mod.grid(*args, rows=(lo, lo + 8))
    assert_parity(got[lo:lo + 8], ref, "cell order, row band")
    assert_parity(got0[lo:lo + 8], ref, "input order, row band")


def _gpu_degrid_cell_order(N, S, O, W, P, uvw, wts, kernel, grid, tuning=None):
    import torch
    from paper_1605_07023_b200 import binding
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    try:
        plan.set_samples(uvw.shape[0])
        plan.set_sample_order(1)
        if tuning:
            plan.set_tuning(**tuning)
        plan.allocate_workspace(dev)
        assert plan.info()["sample_order"] == 1
        out = plan.degrid(torch.from_numpy(uvw).to(dev), torch.from_numpy(wts).to(dev),
                          torch.from_numpy(kernel).to(dev), torch.from_numpy(grid.astype(np.complex64)).to(dev))
        torch.cuda.synchronize()
        launches = plan.last_launches()
        return out.cpu().numpy(), launches
    finally:
        plan.destroy()


@pytest.mark.parametrize("S,P,W", [(7, 1, 3), (8, 4, 3), (16, 1, 3), (16, 2, 3), (32, 4, 3), (12, 4, 3), (40, 1, 3),
                                   (64, 4, 2), (128, 1, 2), (16, 1, 700)])
def test_degrid_in_cell_order(oracle_mod, S, P, W):
    # degridding walks the samples in cell order too: every result must come back to ITS sample's place (the index
    # travels in the record), skipped samples get exact zeros; tolerances as in tests/test_gpu_degrid.py (DESIGN R20)
    N, O, n = (192 if S <= 40 else 384), 4, 9_973
    uvw, _, wts, kernel = synth.random_problem(8100 + S + P, n, N, S, O, W, P, spread=0.52)
    uvw[100:110, 0] = np.nan
    rng = np.random.default_rng(S)
    grid = (rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))).astype(np.complex64)
    ref = oracle_mod.degrid(N, S, O, W, P, uvw, wts, kernel, grid)
    got, launches = _gpu_degrid_cell_order(N, S, O, W, P, uvw, wts, kernel, grid)
    got = got.astype(np.complex128)
    assert launches >= 6, launches                               # the sort's five kernels + the degridding kernel
    q = oracle_mod.quantise(N, S, O, W, uvw)
    assert (q["valid"] == 0).sum() > 10
    assert not got[q["valid"] == 0].any()
    scale = np.sqrt(np.mean(np.abs(ref[q["valid"] == 1]) ** 2))
    assert np.abs(got - ref).max() <= 2e-5 * scale * max(1.0, S / 8)
    assert np.linalg.norm(got - ref) <= 1e-5 * np.linalg.norm(ref)


def test_adjoint_identity_in_cell_order(oracle_mod):
    # <grid(V), G> = <V, degrid(G)> (pin P7) on the CUDA pair, both in cell order
    N, S, O, W, P, n = 256, 8, 8, 2, 4, 40_001
    uvw, vis, wts, kernel = synth.random_problem(8300, n, N, S, O, W, P, spread=0.45, walk=0.7)
    rng = np.random.default_rng(3)
    G = (rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))).astype(np.complex64)
    gridded, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, tuning=dict(sample_order=1))
    assert info["sample_order"] == 1
    degridded, _ = _gpu_degrid_cell_order(N, S, O, W, P, uvw, wts, kernel, G)
    lhs = np.vdot(gridded.astype(np.complex128), G.astype(np.complex128))          # as in tests/test_gpu_degrid.py
    rhs = np.vdot(vis.astype(np.complex128), degridded.astype(np.complex128))
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs)


@pytest.mark.parametrize("P", [1, 4])
def test_cell_order_kept_across_calls(oracle_mod, P):
    # grid_plan_set_sample_order(plan, 2): the first call sorts, later calls with the SAME uvw and weights reuse the
    # sorted records (one launch), whatever the visibilities are; degridding shares them; changing the samples re-sorts
    import torch
    from paper_1605_07023_b200 import binding
    N, S, O, W, n = 160, 8, 4, 2, 30_011
    uvw, vis, wts, kernel = synth.random_problem(8700 + P, n, N, S, O, W, P, spread=0.5, walk=1.3)
    uvw[500:520, 0] = np.nan
    vis2 = (vis * (0.3 - 0.7j) + 1.0).astype(np.complex64)
    dev = torch.device("cuda:0")
    d = {k: torch.from_numpy(np.ascontiguousarray(v)).to(dev) for k, v in
         dict(uvw=uvw, vis=vis, vis2=vis2, wts=wts, kernel=kernel).items()}
    plan = binding.GridPlan(N, S, O, W, P)
    try:
        plan.set_samples(n)
        plan.set_sample_order(2)
        plan.allocate_workspace(dev)
        assert plan.info()["sample_order"] == 1
        g1 = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
        plan.execute(d["uvw"], d["vis"], d["wts"], d["kernel"], g1)
        assert plan.last_launches() == 6
        g2 = torch.zeros_like(g1)
        plan.execute(d["uvw"], d["vis2"], d["wts"], d["kernel"], g2)
        assert plan.last_launches() == 1                          # the gridding kernel alone
        torch.cuda.synchronize()
        assert_parity(g1.cpu().numpy(), oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel), "first call")
        assert_parity(g2.cpu().numpy(), oracle_mod.grid(N, S, O, W, P, uvw, vis2, wts, kernel), "kept order, new visibilities")
        # degridding walks the same records
        rng = np.random.default_rng(P)
        G = (rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))).astype(np.complex64)
        out = plan.degrid(d["uvw"], d["wts"], d["kernel"], torch.from_numpy(G).to(dev))
        assert plan.last_launches() <= 2, plan.last_launches()    # (+ a memset-free kernel only; no sort)
        torch.cuda.synchronize()
        ref = oracle_mod.degrid(N, S, O, W, P, uvw, wts, kernel, G)
        got = out.cpu().numpy().astype(np.complex128)
        assert np.linalg.norm(got - ref) <= 1e-5 * np.linalg.norm(ref)
        # new samples: the records are dropped and rebuilt
        m = n - 1001
        plan.set_samples(m)
        plan.allocate_workspace(dev)
        g3 = torch.zeros_like(g1)
        plan.execute(d["uvw"][:m].contiguous(), d["vis"][:m].contiguous(), d["wts"][:m].contiguous(), d["kernel"], g3)
        assert plan.last_launches() == 6
        torch.cuda.synchronize()
        assert_parity(g3.cpu().numpy(), oracle_mod.grid(N, S, O, W, P, uvw[:m], vis[:m], wts[:m], kernel), "after set_samples")
    finally:
        plan.destroy()


@pytest.mark.parametrize("S,P,W,per_pol", [(8, 4, 2, False), (8, 1, 3, False), (16, 1, 2, False), (32, 4, 1, False),
                                           (16, 2, 2, True), (8, 4, 1, True)])
def test_dense_gcf_in_cell_order(oracle_mod, S, P, W, per_pol):
    # grid_execute_dense / grid_execute_dense_pol walk the sorted records too (one polarisation: the record carries
    # the pre-weighted visibility)
    import torch
    from paper_1605_07023_b200 import binding
    N, O, n = 200, 3, 12_007
    uvw, vis, wts, _ = synth.random_problem(8900 + S + P, n, N, S, O, W, P, spread=0.5, walk=1.2)
    uvw[10:20, 1] = np.nan
    vis[10:20] = np.inf
    rng = np.random.default_rng(S * 7 + P)
    shape = ((P,) if per_pol else ()) + (W, O, O, S, S)
    k2 = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)).astype(np.complex64)
    ref = (oracle_mod.grid_dense_pol if per_pol else oracle_mod.grid_dense)(N, S, O, W, P, uvw, vis, wts, k2)
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    try:
        plan.set_samples(n)
        plan.set_sample_order(1)
        plan.allocate_workspace(dev)
        grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
        call = plan.execute_dense_pol if per_pol else plan.execute_dense
        call(torch.from_numpy(uvw).to(dev), torch.from_numpy(np.ascontiguousarray(vis)).to(dev).reshape(n, P),
             torch.from_numpy(wts).to(dev), torch.from_numpy(k2).to(dev), grid)
        torch.cuda.synchronize()
        assert plan.last_launches() == 6, plan.last_launches()      # the sort's five kernels + the dense kernel
        assert_parity(grid.cpu().numpy(), ref, f"dense in cell order S={S} P={P} W={W} per_pol={per_pol}")
    finally:
        plan.destroy()


def test_cell_order_random_shapes(oracle_mod):
    # 30 seeded random problems: supports 3..64 (most not powers of two), 1/2/4 polarisations, oversampling 1..8,
    # 1..5 planes, grids from the smallest the warp kernel takes, 1..60001 samples (fewer than a batch, a chunk, a
    # warp), random walks from none to 5 cells per sample, some coordinates non-finite -- gridding (modes 1 and 2)
    # and degridding in cell order against the oracle
    import torch
    from paper_1605_07023_b200 import binding
    rng = np.random.default_rng(20260511)
    dev = torch.device("cuda:0")
    for it in range(30):
        S = int(rng.choice([3, 4, 5, 7, 8, 8, 9, 12, 16, 17, 24, 32, 33, 40, 64]))
        P = int(rng.choice([1, 2, 4]))
        O = int(rng.choice([1, 2, 3, 4, 8]))
        W = int(rng.choice([1, 1, 2, 5]))
        Sk = 1 << (S - 1).bit_length()
        N = int(rng.integers(2 * Sk + 1, max(2 * Sk + 2, 600 if S <= 16 else 300)))
        n = int(rng.choice([1, 2, 3, 31, 33, 127, 1000, 4097, 20011, 60001]))
        uvw, vis, wts, kernel = synth.random_problem(int(rng.integers(1 << 30)), n, N, S, O, W, P,
                                                     spread=float(rng.choice([0.3, 0.5, 0.6])),
                                                     walk=float(rng.choice([0.0, 0.2, 1.5, 5.0])))
        if n > 10 and rng.random() < 0.5:
            k = rng.integers(0, n, size=max(1, n // 50))
            uvw[k, int(rng.integers(0, 3))] = rng.choice([np.nan, np.inf, -np.inf, 1e30])
        what = f"case {it}: S={S} P={P} O={O} W={W} N={N} n={n}"
        ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
        got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, tuning=dict(sample_order=int(rng.choice([1, 2]))))
        assert info["sample_order"] == 1, what
        if np.abs(ref).max() == 0:
            assert not got.any(), what
        else:
            assert_parity(got, ref, what)
        G = (rng.standard_normal((N, N, P)) + 1j * rng.standard_normal((N, N, P))).astype(np.complex64)
        out, _ = _gpu_degrid_cell_order(N, S, O, W, P, uvw, wts, kernel, G)
        dref = oracle_mod.degrid(N, S, O, W, P, uvw, wts, kernel, G)
        if np.linalg.norm(dref) == 0:
            assert not out.any(), what
        else:
            assert np.linalg.norm(out - dref) <= 1e-5 * np.linalg.norm(dref), what
