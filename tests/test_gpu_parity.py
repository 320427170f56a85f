"""-m gpu: the CUDA path (through the C ABI binding) against the float64 oracle, element by element,
on the same seeded inputs.  Integer work (step a1) must be bit-exact; FP32 grids must satisfy
rel-L2 <= 1e-5 and max-abs <= 1e-4 * max|grid| (BASELINE.json:north_star; R20)."""
import numpy as np
import pytest

from paper_1605_07023_b200 import synth
from gpu_util import assert_parity, run_gpu

pytestmark = pytest.mark.gpu


def _quantise_gpu(N, S, O, W, uvw):
    import torch
    from paper_1605_07023_b200 import binding
    plan = binding.GridPlan(N, S, O, W, 1)
    try:
        out = plan.quantise(torch.from_numpy(np.ascontiguousarray(uvw)).cuda())
        torch.cuda.synchronize()
        return out.cpu().numpy()
    finally:
        plan.destroy()


def _check_quantise(oracle_mod, N, S, O, W, uvw):
    got = _quantise_gpu(N, S, O, W, uvw)
    ref = oracle_mod.quantise(N, S, O, W, uvw)
    for col, key in enumerate(("i0", "j0", "su", "sv", "wp", "valid")):
        assert np.array_equal(got[:, col], ref[key].astype(np.int32)), key
    return int(ref["valid"].sum())


@pytest.mark.parametrize("N,S,O,W", [(512, 7, 8, 1), (2048, 8, 8, 1), (4096, 16, 8, 32), (64, 5, 3, 2),
                                     (33, 4, 5, 1), (16, 1, 1, 1), (8192, 32, 8, 16)])
def test_quantise_bit_exact_random_and_ties(oracle_mod, N, S, O, W):
    rng = np.random.default_rng(N + S)
    n = 200_003
    uvw = np.empty((n, 3), np.float32)
    uvw[:, :2] = rng.uniform(-0.55 * N, 0.55 * N, (n, 2))
    # exact ties between oversampled points, cell boundaries, tiny and huge values, non-finite
    ties = ((rng.integers(-N * O, N * O, n // 4) + 0.5) / O).astype(np.float32)
    uvw[: n // 4, 0] = ties
    uvw[n // 4: n // 2, 1] = np.round(uvw[n // 4: n // 2, 1])
    uvw[:, 2] = rng.uniform(-1.5 * W, 1.5 * W, n)
    uvw[::97, 2] = np.round(uvw[::97, 2])
    special = np.array([np.nan, np.inf, -np.inf, 1e30, -1e30, 1e-40, -1e-40, 0.0, -0.0], np.float32)
    for k, v in enumerate(special):
        uvw[1000 + 3 * k, 0] = v
        uvw[1001 + 3 * k, 1] = v
        uvw[1002 + 3 * k, 2] = v
    nv = _check_quantise(oracle_mod, N, S, O, W, uvw)
    assert 0 < nv < n


def test_quantise_bit_exact_cfg0(oracle_mod):
    wl = synth.make_workload(synth.get_config("cfg0"))
    c = wl.cfg
    assert _check_quantise(oracle_mod, c.grid_size, c.support, c.oversample, c.n_wplanes, wl.uvw) == c.n_vis


def test_cfg0_full_parity(oracle_mod):
    wl = synth.make_workload(synth.get_config("cfg0"))
    c = wl.cfg
    ref = oracle_mod.grid(c.grid_size, c.support, c.oversample, c.n_wplanes, c.n_pol, wl.uvw, wl.vis,
                          wl.weights, wl.kernel)
    for layout in (None, (c.n_baselines, c.n_times, c.n_chan)):
        got, info = run_gpu(c.grid_size, c.support, c.oversample, c.n_wplanes, c.n_pol, wl.uvw, wl.vis,
                            wl.weights, wl.kernel, layout=layout)
        rel, mx = assert_parity(got, ref, f"cfg0 layout={layout}")
        print(f"cfg0 layout={layout}: rel={rel:.2e} max={mx:.2e} {info}")


COMBOS = [(1, 1, 1), (2, 1, 1), (2, 2, 1), (4, 1, 1), (4, 2, 1), (4, 4, 1), (8, 2, 1), (8, 4, 1),
          (1, 1, 2), (2, 1, 2), (2, 2, 2), (4, 2, 2), (4, 4, 2),
          (1, 1, 4), (2, 1, 4), (2, 2, 4), (4, 1, 4), (4, 2, 4)]


@pytest.mark.parametrize("cu,cv,P", COMBOS)
@pytest.mark.parametrize("S", [7, 8])
def test_every_coarsening_block(oracle_mod, cu, cv, P, S):
    # several chunks per team, a ragged tail (n not a multiple of batch, chunk or 4), samples that
    # fall off the grid, two planes
    N, O, W, n = 96, 8, 2, 30_001
    uvw, vis, wts, kernel = synth.random_problem(100 * cu + 10 * cv + P + S, n, N, S, O, W, P,
                                                 spread=0.5, walk=1.2)
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel,
                        tuning=dict(variant=1, cu=cu, cv=cv, threads_per_cta=128, batch=32, chunk=200))
    assert (info["variant"], info["cu"], info["cv"]) == (1, cu, cv)
    assert_parity(got, ref, f"C={cu}x{cv} P={P} S={S}")


# every instantiated block of the warp kernel (= the autotuner's candidates)
WARP = [(2, 2, 1), (4, 2, 1), (4, 4, 1), (8, 4, 1), (2, 2, 2), (4, 2, 2), (4, 4, 2), (2, 2, 4), (4, 2, 4)]


@pytest.mark.parametrize("cu,cv,P", WARP)
@pytest.mark.parametrize("S", [4, 8, 16, 32])
def test_every_warp_block(oracle_mod, cu, cv, P, S):
    # warp-autonomous kernel (variant 3): teams of 1..1024 threads (several teams per warp up to a
    # whole CTA per team), ragged tail, samples off the grid, jumps larger than the support, 3 planes
    if cu > S or cv > S:
        pytest.skip("block larger than the support")
    N, O, W, n = 128, 4, 3, 20_003
    uvw, vis, wts, kernel = synth.random_problem(2000 + 100 * cu + 10 * cv + P + S, n, N, S, O, W, P,
                                                 spread=0.5, walk=1.5)
    uvw[5000:5100, :2] = np.random.default_rng(S).uniform(-60, 60, (100, 2))    # big jumps
    uvw[7000:7010, 0] = np.nan
    vis[7000:7010] = np.inf
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    for batch, chunk in ((32, 300), (8, 64)):
        got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel,
                            tuning=dict(variant=3, cu=cu, cv=cv, threads_per_cta=1024, batch=batch, chunk=chunk))
        assert (info["variant"], info["cu"], info["cv"], info["bin_u"]) == (3, cu, cv, S)
        assert_parity(got, ref, f"warp C={cu}x{cv} P={P} S={S} batch={batch} {info}")


@pytest.mark.parametrize("cu,cv", [(2, 2), (4, 2), (4, 4)])
@pytest.mark.parametrize("S", [4, 8, 16, 32])
def test_warp_block_pol_split(oracle_mod, cu, cv, S):
    # 4 polarisations spread over lane pairs (grid_plan_set_pol_split): same result as the oracle
    if cu > S or cv > S:
        pytest.skip("block larger than the support")
    N, O, W, P, n = 128, 4, 3, 4, 20_003
    uvw, vis, wts, kernel = synth.random_problem(3000 + 10 * cu + cv + S, n, N, S, O, W, P, spread=0.5, walk=1.5)
    uvw[5000:5100, :2] = np.random.default_rng(S).uniform(-60, 60, (100, 2))
    uvw[7000:7010, 0] = np.nan
    vis[7000:7010] = np.inf
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel,
                        tuning=dict(pol_split=2, variant=3, cu=cu, cv=cv, threads_per_cta=1024, batch=16, chunk=200))
    assert (info["variant"], info["cu"], info["cv"]) == (3, cu, cv)
    assert_parity(got, ref, f"pol-split C={cu}x{cv} S={S} {info}")


@pytest.mark.parametrize("S,P,cu,cv", [(1, 1, 1, 1), (2, 4, 2, 1), (3, 1, 2, 2), (4, 1, 4, 2), (5, 2, 2, 2),
                                       (16, 1, 4, 4), (16, 4, 2, 2), (32, 1, 8, 4), (32, 4, 4, 2), (13, 1, 4, 4)])
def test_supports(oracle_mod, S, P, cu, cv):
    N, O, W, n = 160, 4, 3, 12_345
    uvw, vis, wts, kernel = synth.random_problem(7 * S + P, n, N, S, O, W, P, spread=0.48, walk=2.0)
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel,
                        tuning=dict(variant=1, cu=cu, cv=cv, threads_per_cta=512))
    assert_parity(got, ref, f"S={S} P={P} {info}")


def test_default_tuning_all_config_shapes(oracle_mod):
    # the (S, P, planes) of every BASELINE config with the plan's own default tuning, shrunk arrays
    for name in ["cfg0", "cfg1", "cfg2", "cfg3"] + [f"cfg4_S{s}_P{p}" for s in (4, 8, 16, 32) for p in (1, 4)]:
        cfg = synth.shrink(synth.get_config(name), n_ant=10, n_times=24, n_chan=12, grid_size=512)
        wl = synth.make_workload(cfg)
        ref = oracle_mod.grid(cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol,
                              wl.uvw, wl.vis, wl.weights, wl.kernel)
        got, info = run_gpu(cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol,
                            wl.uvw, wl.vis, wl.weights, wl.kernel,
                            layout=(cfg.n_baselines, cfg.n_times, cfg.n_chan))
        rel, mx = assert_parity(got, ref, name)
        print(f"{name}: rel={rel:.2e} max={mx:.2e} C={info['cu']}x{info['cv']}")


@pytest.mark.parametrize("mode", [-1, 0, 1])
@pytest.mark.parametrize("n_ant,n_times,n_chan,tc", [(9, 37, 13, 16), (7, 5, 64, 16), (12, 64, 3, 8), (6, 33, 40, 32)])
def test_traversal_modes(oracle_mod, mode, n_ant, n_times, n_chan, tc):
    # ragged time blocks (n_times % tc != 0), channel counts that are not a multiple of the batch
    # columns, fewer time steps than one block
    for name in ("cfg1", "cfg2"):
        cfg = synth.shrink(synth.get_config(name), n_ant=n_ant, n_times=n_times, n_chan=n_chan, grid_size=384)
        wl = synth.make_workload(cfg)
        ref = oracle_mod.grid(cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol,
                              wl.uvw, wl.vis, wl.weights, wl.kernel)
        got, info = run_gpu(cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol,
                            wl.uvw, wl.vis, wl.weights, wl.kernel,
                            layout=(cfg.n_baselines, cfg.n_times, cfg.n_chan),
                            tuning=dict(traversal=mode, time_block=tc, threads_per_cta=128))
        assert (info["traversal"], info["time_block"]) == (mode, tc)
        assert_parity(got, ref, f"{name} mode={mode}")


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("name,ps", [("cfg1", 1), ("cfg3", 2), ("cfg2", 1)])
def test_sorted_chunk_queue(oracle_mod, name, ps, mode):
    # chunk ids sorted by grid tile (grid_plan_set_chunk_order): same sum, both traversal modes, small chunks
    cfg = synth.shrink(synth.get_config(name), n_ant=14, n_times=40, n_chan=24, grid_size=1024)
    wl = synth.make_workload(cfg)
    ref = oracle_mod.grid(cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol,
                          wl.uvw, wl.vis, wl.weights, wl.kernel)
    tuning = dict(chunk_order=1, traversal=mode, chunk=64, batch=16)
    if cfg.n_pol == 4:
        tuning["pol_split"] = ps
    got, info = run_gpu(cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol,
                        wl.uvw, wl.vis, wl.weights, wl.kernel,
                        layout=(cfg.n_baselines, cfg.n_times, cfg.n_chan), tuning=tuning)
    assert info["chunk_order"] == 1 and info["launches"] == 5
    assert_parity(got, ref, f"{name} sorted queue mode={mode}")


@pytest.mark.parametrize("cu,cv,P,W", [(8, 4, 1, 2), (4, 4, 1, 2), (4, 2, 1, 3), (4, 2, 4, 2), (4, 4, 2, 2), (4, 2, 2, 2),
                                       (8, 4, 1, 40), (4, 2, 4, 40)])
@pytest.mark.parametrize("mode", [0, 1])
def test_support_64(oracle_mod, cu, cv, P, W, mode):
    # S = 64 (the paper's bin 64): 64-bit moved masks, teams of 128-1024 threads synchronised by named
    # barriers; tap table in shared memory (W <= 3) and in global memory (W = 40); jumps beyond the support
    S, O = 64, 4
    cfg = synth.shrink(synth.get_config("cfg1"), n_ant=7, n_times=21, n_chan=9, grid_size=640)
    rng = np.random.default_rng(cu + 10 * cv + P)
    uvw = synth.make_uvw(cfg, rng)
    n = uvw.shape[0]
    uvw[:, 2] = rng.uniform(0, W, n)
    uvw[30:40, :2] = rng.uniform(-250, 250, (10, 2))
    uvw[40:45, 0] = np.nan
    vis = (rng.standard_normal((n, P)) + 1j * rng.standard_normal((n, P))).astype(np.complex64)
    wts = rng.uniform(0.5, 1, n).astype(np.float32)
    kernel = (rng.standard_normal((W, O, S)) + 1j * rng.standard_normal((W, O, S))).astype(np.complex64)
    N = cfg.grid_size
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, layout=(cfg.n_baselines, cfg.n_times, cfg.n_chan),
                        tuning=dict(variant=3, cu=cu, cv=cv, threads_per_cta=1024, batch=16, chunk=64, traversal=mode, time_block=8))
    assert (info["variant"], info["cu"], info["cv"], info["bin_u"]) == (3, cu, cv, 64)
    assert info["taps_global"] == (1 if W == 40 else 0)
    assert_parity(got, ref, f"S=64 C={cu}x{cv} P={P} W={W} mode={mode} {info}")


@pytest.mark.parametrize("cu,cv,P,W", [(8, 4, 1, 2), (4, 4, 1, 2), (4, 2, 4, 2), (4, 4, 2, 2), (8, 4, 1, 40), (4, 2, 4, 40)])
@pytest.mark.parametrize("mode", [0, 1])
def test_support_128_tiled(oracle_mod, cu, cv, P, W, mode):
    # S = 128 (the paper's largest bin): the bin is split into 2 x 2 tiles of 64 x 64 positions, one team per
    # tile, every tile re-reading the chunk; jumps beyond a tile and beyond the support
    S, O = 128, 2
    cfg = synth.shrink(synth.get_config("cfg1"), n_ant=6, n_times=19, n_chan=7, grid_size=768)
    rng = np.random.default_rng(3 * cu + 10 * cv + P)
    uvw = synth.make_uvw(cfg, rng)
    n = uvw.shape[0]
    uvw[:, 2] = rng.uniform(0, W, n)
    uvw[30:40, :2] = rng.uniform(-300, 300, (10, 2))
    uvw[50:60, :2] = uvw[49, :2] + rng.uniform(-90, 90, (10, 2))      # jumps around one tile width
    uvw[40:45, 0] = np.nan
    vis = (rng.standard_normal((n, P)) + 1j * rng.standard_normal((n, P))).astype(np.complex64)
    wts = rng.uniform(0.5, 1, n).astype(np.float32)
    kernel = (rng.standard_normal((W, O, S)) + 1j * rng.standard_normal((W, O, S))).astype(np.complex64)
    N = cfg.grid_size
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, layout=(cfg.n_baselines, cfg.n_times, cfg.n_chan),
                        tuning=dict(variant=3, cu=cu, cv=cv, threads_per_cta=1024, batch=16, chunk=64, traversal=mode, time_block=8))
    assert (info["variant"], info["cu"], info["cv"], info["bin_u"]) == (3, cu, cv, 128)
    assert_parity(got, ref, f"S=128 C={cu}x{cv} P={P} W={W} mode={mode} {info}")


@pytest.mark.parametrize("S,W,P", [(16, 700, 1), (32, 300, 4), (8, 1500, 4), (32, 1229, 1), (4, 4000, 1), (16, 520, 2)])
def test_tap_table_beyond_shared_memory(oracle_mod, S, W, P):
    # many w-planes (the paper: 1229 per slice): the plan switches to the kernels that read the
    # taps from global memory; same result as the oracle, also through the compressed entry point
    N, O, n = 192, 8, 25_001
    uvw, vis, wts, kernel = synth.random_problem(500 + S + P, n, N, S, O, W, P, spread=0.5, walk=0.7)
    assert len(np.unique(np.floor(uvw[:, 2]))) > 0.2 * min(W, n)             # planes all over the table
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel)
    assert info["variant"] == 3 and info["taps_global"] == 1 and info["launches"] == 3
    assert_parity(got, ref, f"global taps S={S} W={W} P={P} {info}")


def test_inconsistent_layout_hint_is_ignored(oracle_mod):
    cfg = synth.shrink(synth.get_config("cfg1"), n_ant=8, n_times=16, n_chan=8, grid_size=256)
    wl = synth.make_workload(cfg)
    ref = oracle_mod.grid(cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol,
                          wl.uvw, wl.vis, wl.weights, wl.kernel)
    got, _ = run_gpu(cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol,
                     wl.uvw, wl.vis, wl.weights, wl.kernel, layout=(3, 5, 7), tuning=dict(traversal=1))
    assert_parity(got, ref, "bad layout")


@pytest.mark.parametrize("S,P", [(64, 4), (128, 1), (100, 2), (48, 4), (7, 1), (13, 4), (3, 2), (40, 1), (5, 4)])
def test_large_supports_have_a_path(oracle_mod, S, P):
    # the ABI accepts supports up to 128 (the paper's bins: 32, 64, 128).  Supports that are not powers of two run
    # on the warp kernel too, zero-padded to the next power of two (pin P14): never on the
    # one-atomic-per-update kernel.  Samples near both edges of the grid exercise both padded copies of the tap rows.
    N, O, W, n = 512, 2, 2, 3_001
    uvw, vis, wts, kernel = synth.random_problem(900 + S + P, n, N, S, O, W, P, spread=0.45, walk=0.5)
    edge = N // 2 - S // 2 - 1
    uvw[100:140, 0] = np.linspace(edge - 3, edge + 2, 40)      # upper edge in u: some valid, some off the grid
    uvw[200:240, 1] = np.linspace(edge - 3, edge + 2, 40)
    uvw[300:340, :2] = -np.linspace(edge - 3, edge + 2, 40)[:, None]
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, info = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel)
    print(S, P, info)
    assert info["variant"] == 3
    assert_parity(got, ref, f"S={S} P={P} {info}")


def test_scatter_variant(oracle_mod):
    N, S, O, W, P, n = 128, 6, 4, 2, 4, 5001
    uvw, vis, wts, kernel = synth.random_problem(42, n, N, S, O, W, P, spread=0.52)
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    got, _ = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, tuning=dict(variant=0))
    assert_parity(got, ref, "scatter")


def test_edge_cases(oracle_mod):
    import torch
    from paper_1605_07023_b200 import binding
    N, S, O, W, P = 64, 8, 8, 1, 4
    kernel = synth.random_problem(1, 1, N, S, O, W, P)[3]
    # n_vis = 0: no-op, grid untouched (R23)
    init = (np.arange(N * N * P, dtype=np.float32).reshape(N, N, P) * (1 + 1j)).astype(np.complex64)
    got, info = run_gpu(N, S, O, W, P, np.zeros((0, 3), np.float32), np.zeros((0, P), np.complex64),
                        np.zeros(0, np.float32), kernel, grid_init=init)
    assert np.array_equal(got, init) and info["launches"] == 0
    # all samples invalid: grid untouched
    uvw = np.full((100, 3), np.nan, np.float32)
    uvw[50:] = 1e6
    got, _ = run_gpu(N, S, O, W, P, uvw, np.ones((100, P), np.complex64), np.ones(100, np.float32), kernel,
                     grid_init=init)
    assert np.array_equal(got, init)
    # accumulation into a non-zero grid (R10) and Inf visibilities on skipped samples must not leak
    uvw, vis, wts, _ = synth.random_problem(3, 999, N, S, O, W, P, spread=0.7)
    bad = oracle_mod.quantise(N, S, O, W, uvw)["valid"] == 0
    assert bad.any()
    vis[bad] = np.inf
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel) + init.astype(np.complex128)
    got, _ = run_gpu(N, S, O, W, P, uvw, vis, wts, kernel, grid_init=init)
    assert_parity(got, ref, "accumulate")
    # single sample; footprint touching the grid corner; S = N
    for (n_, s_, u, v) in [(64, 8, -28.0, -28.0), (64, 8, 27.4, 27.4), (8, 8, -1.0, -1.0)]:
        k = synth.random_problem(5, 1, n_, s_, 2, 1, 1)[3]
        one = np.array([[u, v, 0.0]], np.float32)
        ref = oracle_mod.grid(n_, s_, 2, 1, 1, one, np.ones((1, 1), np.complex64), np.ones(1, np.float32), k)
        assert np.count_nonzero(ref) == s_ * s_
        got, _ = run_gpu(n_, s_, 2, 1, 1, one, np.ones((1, 1), np.complex64), np.ones(1, np.float32), k)
        assert_parity(got, ref, f"single {n_} {s_}")
    # error behaviour: missing set_samples / workspace, CPU tensors
    plan = binding.GridPlan(N, S, O, W, P)
    t = torch.zeros((4, 3), device="cuda")
    with pytest.raises(binding.GridError):
        plan.execute(t, t, t, t, t)
    plan.set_samples(4)
    with pytest.raises(binding.GridError):
        plan.execute(torch.zeros((4, 3), device="cuda"), torch.zeros((4, P), dtype=torch.complex64, device="cuda"),
                     torch.zeros(4, device="cuda"), torch.zeros((W, O, S), dtype=torch.complex64, device="cuda"),
                     torch.zeros((N, N, P), dtype=torch.complex64, device="cuda"))
    with pytest.raises(TypeError):                    # host memory is rejected: no CPU fallback
        plan.execute(torch.zeros((4, 3)), torch.zeros((4, P), dtype=torch.complex64, device="cuda"),
                     torch.zeros(4, device="cuda"), torch.zeros((W, O, S), dtype=torch.complex64, device="cuda"),
                     torch.zeros((N, N, P), dtype=torch.complex64, device="cuda"))
    plan.destroy()


def test_repeat_execute_accumulates(oracle_mod):
    import torch
    from paper_1605_07023_b200 import binding
    N, S, O, W, P, n = 128, 8, 8, 2, 1, 20_000
    uvw, vis, wts, kernel = synth.random_problem(77, n, N, S, O, W, P, spread=0.4, walk=1.0)
    ref = oracle_mod.grid(N, S, O, W, P, uvw, vis, wts, kernel)
    plan = binding.GridPlan(N, S, O, W, P)
    plan.set_samples(n)
    plan.allocate_workspace()
    grid = torch.zeros((N, N, P), dtype=torch.complex64, device="cuda")
    args = [torch.from_numpy(a).cuda() for a in (uvw, vis, wts, kernel)]
    for _ in range(3):
        plan.execute(*args, grid)
    torch.cuda.synchronize()
    plan.destroy()
    assert_parity(grid.cpu().numpy(), 3 * ref, "3x execute")


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg0"])
def test_autotuned_plan_stays_in_parity(oracle_mod, name):
    # grid_plan_autotune: times every candidate block on a synthetic data set, installs the fastest;
    # the tuned plan must give the oracle's grid, and the result table must cover every candidate
    import torch
    from paper_1605_07023_b200 import binding
    cfg = synth.shrink(synth.get_config(name), n_ant=12, n_times=40, n_chan=16, grid_size=512)
    wl = synth.make_workload(cfg)
    N, S, O, W, P = cfg.grid_size, cfg.support, cfg.oversample, cfg.n_wplanes, cfg.n_pol
    ref = oracle_mod.grid(N, S, O, W, P, wl.uvw, wl.vis, wl.weights, wl.kernel)
    dev = torch.device("cuda:0")
    plan = binding.GridPlan(N, S, O, W, P)
    plan.set_samples(cfg.n_vis)
    plan.set_layout(cfg.n_baselines, cfg.n_times, cfg.n_chan)
    cands = plan.autotune_candidates()
    table = plan.autotune(n_samples=1 << 17, seed=3)
    assert [c for c, _ in table] == cands and all(us > 0 for _, us in table), table
    i = plan.info()
    best = min(table, key=lambda e: e[1])[0]
    assert (i["cu"], i["cv"], i["pol_split"]) == best
    plan.allocate_workspace(dev)
    grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
    plan.execute(*(torch.from_numpy(a).to(dev) for a in (wl.uvw, wl.vis, wl.weights, wl.kernel)), grid)
    torch.cuda.synchronize()
    plan.destroy()
    assert_parity(grid.cpu().numpy(), ref, f"autotuned {name}: {best} of {table}")
