"""-m "not gpu": the C-ABI library loads, exports every symbol include/grid.h declares, and its host
logic (argument validation, bin / team derivation, workspace sizing) behaves as documented.
No compute entry point is called here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    import __graft_entry__ as entry
    entry.build()
    from paper_1605_07023_b200 import binding as b
    return b


def test_header_symbols_are_exported(binding):
    header = open(os.path.join(ROOT, "include", "grid.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(grid_[a-z_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    lib = ctypes.CDLL(binding.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def test_no_torch_types_in_header():
    header = open(os.path.join(ROOT, "include", "grid.h")).read()
    assert "torch" not in header.lower().replace("pytorch", "") and "at::" not in header


def test_plan_validation(binding):
    for args in [(0, 8, 8, 1, 4), (2048, 0, 8, 1, 4), (2048, 8, 0, 1, 4), (2048, 8, 8, 0, 4), (2048, 8, 8, 1, 3),
                 (4, 8, 8, 1, 1), (40000, 8, 8, 1, 1), (2048, 8, 8, 70000, 1)]:
        with pytest.raises(binding.GridError):
            binding.GridPlan(*args)
        assert binding.grid_last_error() != ""


@pytest.mark.parametrize("S,P", [(7, 1), (8, 4), (16, 1), (8, 1), (4, 1), (4, 4), (16, 4), (32, 1), (32, 4), (1, 1), (12, 4), (100, 1), (3, 2)])
def test_default_plan_geometry(binding, S, P):
    plan = binding.GridPlan(4096, S, 8, 16, P)
    i = plan.info()
    if i["variant"] == 3:
        # bin == support rounded up to a power of two (zero-padded taps); owned positions S/C
        # apart (north_star: "taken modulo the support")
        sk = 4
        while sk < S:
            sk *= 2
        assert S >= 3 and i["bin_u"] == i["bin_v"] == sk
    else:
        # bin >= S + C - 1, aligned to the block; a team covers the bin exactly
        assert i["bin_u"] % i["cu"] == 0 and i["bin_v"] % i["cv"] == 0
        assert S + i["cu"] - 1 <= i["bin_u"] < S + 2 * i["cu"] - 1
        assert S + i["cv"] - 1 <= i["bin_v"] < S + 2 * i["cv"] - 1
    tile = min(i["bin_u"], 64) if i["variant"] == 3 else i["bin_u"]      # S = 128: a team covers a 64 x 64 tile
    tile_v = min(i["bin_v"], 64) if i["variant"] == 3 else i["bin_v"]
    assert i["team_threads"] == (tile // i["cu"]) * (tile_v // i["cv"]) * max(i["pol_split"], 1)
    assert 1 <= i["teams_per_cta"] <= i["threads_per_cta"] // i["team_threads"]
    assert i["cu"] * i["cv"] * P // max(i["pol_split"], 1) <= 32
    assert i["smem_bytes"] <= 227 * 1024
    plan.destroy()


def test_workspace_and_tuning(binding):
    plan = binding.GridPlan(2048, 8, 8, 1, 4)
    assert plan.workspace_bytes() == 0              # set_samples not called yet
    plan.set_samples(1001)
    head = 256 + 2 * 1024 * 4                       # counters + chunk-order bins
    assert plan.workspace_bytes() == head + 1004 * 16 + ((1001 // 8 + 4096) * 4 + 15) // 16 * 16
    plan.set_samples(0)
    assert plan.workspace_bytes() == head + 4096 * 4
    plan.set_layout(10, 10, 10)
    plan.set_tuning(variant=1, cu=2, cv=2, threads_per_cta=128, batch=32, chunk=512, ctas_per_sm=3)
    i = plan.info()
    assert (i["cu"], i["cv"], i["bin_u"], i["bin_v"], i["team_threads"], i["teams_per_cta"]) == (2, 2, 10, 10, 25, 5)
    assert (i["batch"], i["chunk"], i["ctas_per_sm"]) == (32, 512, 3)
    for bad in [dict(cu=3), dict(threads_per_cta=100), dict(batch=48), dict(cu=4, cv=4),   # 4x4x4 accumulators
                dict(threads_per_cta=32, cu=1, cv=1), dict(batch=1 << 14)]:
        with pytest.raises(binding.GridError) as e:
            plan.set_tuning(**bad)
        assert e.value.code == binding.GRID_ERR_UNSUPPORTED
    assert plan.info() == i                          # failed overrides leave the plan unchanged
    with pytest.raises(binding.GridError):
        plan.set_samples(-1)
    plan.destroy()


def test_compute_calls_reject_host_memory(binding):
    import torch
    plan = binding.GridPlan(64, 8, 8, 1, 1)
    plan.set_samples(4)
    with pytest.raises(TypeError):                   # CPU tensors: no CPU fallback
        plan.execute(torch.zeros(4, 3), torch.zeros(4, 1, dtype=torch.complex64), torch.zeros(4),
                     torch.zeros(1, 8, 8, dtype=torch.complex64), torch.zeros(64, 64, 1, dtype=torch.complex64))
    plan.destroy()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1605_07023_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", text, flags=re.M), f
                assert "gridder_oracle" not in text, f


def test_no_silent_scatter_fallback(binding):
    """Every support in [3, 128] gets the warp kernel (zero-padded to a power of two where needed) for any plane count
    the ABI accepts, tap table in shared or global memory -- never the one-atomic-per-update kernel (variant 0), which
    round 1 fell back to for 1755 of 2688 (S, P, W, O) combinations.  Host logic only: no device needed."""
    bad = []
    for S in list(range(3, 41)) + [48, 63, 64, 65, 100, 127, 128]:
        for P in (1, 2, 4):
            for W, O in ((1, 8), (32, 8), (128, 8), (1229, 8), (16, 4)):
                plan = binding.GridPlan(4096, S, O, W, P)
                i = plan.info()
                plan.destroy()
                if i["variant"] != 3:
                    bad.append((S, P, W, O, i["variant"]))
    assert not bad, bad[:10]
    # the one documented exception: grids smaller than twice the padded support fall back, and say so
    plan = binding.GridPlan(18, 13, 4, 1, 1)
    assert plan.info()["variant"] in (0, 1)
    plan.destroy()


def test_autotune_candidates_host_logic(binding):
    """grid_plan_autotune_candidates ("a range of coarsening factors and work-group sizes"): host logic,
    no device.  The current (default) block comes first; every candidate is a block the plan accepts; polarisation
    splits only with 4 polarisations; supports that do not run the warp kernel have none."""
    for args in [(2048, 8, 8, 1, 4), (4096, 16, 8, 32, 1), (512, 7, 8, 1, 1), (4096, 32, 8, 16, 4), (4096, 64, 8, 16, 2),
                 (4096, 128, 8, 1229, 1), (4096, 12, 4, 3, 2)]:
        plan = binding.GridPlan(*args)
        i = plan.info()
        cands = plan.autotune_candidates()
        assert cands and cands[0] == (i["cu"], i["cv"], i["pol_split"]), (args, cands)
        assert len(set(cands)) == len(cands)
        assert all(ps == 1 or args[4] == 4 for _, _, ps in cands)
        for cu, cv, ps in cands:                       # each one can be installed by hand
            trial = binding.GridPlan(*args)
            try:                                       # split first, then the block -- or the other way round
                if ps != trial.info()["pol_split"]:
                    trial.set_pol_split(ps)
                trial.set_tuning(cu=cu, cv=cv)
            except binding.GridError:
                trial.set_tuning(cu=cu, cv=cv)
                trial.set_pol_split(ps)
            assert (trial.info()["cu"], trial.info()["cv"], trial.info()["pol_split"]) == (cu, cv, ps)
            trial.destroy()
        plan.destroy()
    plan = binding.GridPlan(64, 2, 4, 1, 1)           # support 2: the padded kernel, nothing to tune
    assert plan.autotune_candidates() == []
    plan.destroy()


def test_autotune_needs_a_device(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present: covered by the GPU test")
    plan = binding.GridPlan(2048, 8, 8, 1, 4)
    with pytest.raises(binding.GridError) as e:
        plan.autotune(stream=0)                        # the default stream by handle: torch has no device to ask
    assert e.value.code == binding.GRID_ERR_CUDA       # no CPU fallback, no silent success
    plan.destroy()


def test_sample_order_host_logic(binding):
    # grid_plan_set_sample_order (include/grid.h): the automatic rule, the workspace it needs, the block it selects
    def plan(N, S, P, n, layout=None, W=1):
        p = binding.GridPlan(N, S, 8, W, P)
        p.set_samples(n)
        if layout:
            p.set_layout(*layout)
        return p
    big = 2016 * 256 * 64
    p = plan(2048, 8, 4, big, (2016, 256, 64))
    try:
        assert p.info()["sample_order"] == 1                              # large multi-channel input: cell order
        ws_cell = p.workspace_bytes()
        assert (p.info()["cu"], p.info()["cv"], p.info()["pol_split"]) == (2, 2, 1)
        p.set_sample_order(0)
        assert p.info()["sample_order"] == 0
        ws_input = p.workspace_bytes()
        # 4 bytes per grid cell (+ 1, rounded to the scan tile) + 16 more bytes per record + 4 per rank, and change
        extra = ws_cell - ws_input
        assert 4 * 2048 * 2048 + 20 * big <= extra <= 4 * 2048 * 2048 + 20 * big + (1 << 20), extra
        p.set_sample_order(2)
        assert p.info()["sample_order"] == 1 and p.workspace_bytes() == ws_cell
        with pytest.raises(binding.GridError):
            p.set_sample_order(3)
    finally:
        p.destroy()
    for args, want in (((2048, 8, 4, (1 << 20) - 1), 0),                  # small input: the extra launches do not pay
                       ((2048, 8, 4, 1 << 20), 1),
                       ((8192, 8, 4, 1 << 22), 0),                        # histogram of 67 M cells for 4 M samples
                       ((8192, 8, 4, 1 << 23), 1),
                       ((4096, 32, 4, 64 * 63 // 2 * 3600, (2016, 3600, 1)), 0),   # single-channel tracks (the paper's data)
                       ((4096, 32, 4, 64 * 63 // 2 * 3600), 1),
                       ((4096, 16, 1, 33_030_144, (2016, 128, 128), 32), 1)):
        p = plan(*args)
        try:
            assert p.info()["sample_order"] == want, (args, p.info())
        finally:
            p.destroy()
    # the scatter and padded kernels have no cell order
    p = plan(2048, 8, 4, big)
    try:
        p.set_sample_order(0)
        p.set_tuning(variant=1, cu=2, cv=2, threads_per_cta=256, batch=32, chunk=256)
        with pytest.raises(binding.GridError):
            p.set_sample_order(1)
        assert p.info()["sample_order"] == 0
    finally:
        p.destroy()


def test_build_ptx_quality_check(tmp_path):
    # __graft_entry__.build() looks at the PTX of the product library: nvcc 12.9's split compile emits, at random, a
    # PTX that re-reads kernel parameters at every use (3.4 % slower gridding kernels); the build is repeated until the
    # parameters are read once.  The check itself:
    import __graft_entry__ as entry
    good = ".visible .entry k1(\n.param .align 8 .b8 p[8])\n{\n" + "ld.param.u32 %r1, [p];\n" * 50 + "}\n"
    (tmp_path / "gridder.ptx").write_text(good * 3)
    assert entry._ptx_quality(str(tmp_path)) == 50
    (tmp_path / "gridder.ptx").write_text((good + "ld.param.u64 %rd1, [p];\n" * 170) * 3)
    q = entry._ptx_quality(str(tmp_path))
    assert q == 220 and q > entry.LD_PARAM_PER_KERNEL >= 100
    assert entry._ptx_quality(str(tmp_path / "missing")) is None
