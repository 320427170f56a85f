"""Helpers for the -m gpu parity tests: run the CUDA path through the binding (C ABI) and compare
with the float64 oracle.  Tolerances are BASELINE.json:north_star's (R20)."""
import numpy as np

REL_L2_TOL = 1e-5          # ||g_gpu - g_ref||_2 / ||g_ref||_2
MAX_ABS_TOL = 1e-4         # max |g_gpu - g_ref| / max |g_ref|


def run_gpu(N, S, O, W, P, uvw, vis, weights, kernel, layout=None, tuning=None, grid_init=None):
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
            if "traversal" in tuning or "time_block" in tuning:
                plan.set_traversal(tuning.pop("traversal", -1), tuning.pop("time_block", 0))
            if "chunk_order" in tuning:
                plan.set_chunk_order(tuning.pop("chunk_order"))
            if "sample_order" in tuning:
                plan.set_sample_order(tuning.pop("sample_order"))
            if "pol_split" in tuning:          # before the block: (cu, cv) is validated against it
                plan.set_pol_split(tuning.pop("pol_split"))
            if tuning:
                plan.set_tuning(**tuning)
        plan.allocate_workspace(dev)
        if grid_init is None:
            grid = torch.zeros((N, N, P), dtype=torch.complex64, device=dev)
        else:
            grid = torch.from_numpy(grid_init).to(dev)
        d_uvw = torch.from_numpy(np.ascontiguousarray(uvw)).to(dev).reshape(n, 3)
        d_vis = torch.from_numpy(np.ascontiguousarray(vis)).to(dev).reshape(n, P)
        d_w = torch.from_numpy(np.ascontiguousarray(weights)).to(dev)
        d_k = torch.from_numpy(np.ascontiguousarray(kernel)).to(dev)
        plan.execute(d_uvw, d_vis, d_w, d_k, grid)
        torch.cuda.synchronize()
        info = plan.info()
        info["launches"] = plan.last_launches()
        return grid.cpu().numpy(), info
    finally:
        plan.destroy()


def errors(got, ref):
    got = got.astype(np.complex128)
    diff = got - ref
    nref = np.linalg.norm(ref.ravel())
    rel = np.linalg.norm(diff.ravel()) / nref if nref > 0 else np.linalg.norm(diff.ravel())
    mref = np.abs(ref).max()
    mx = np.abs(diff).max() / mref if mref > 0 else np.abs(diff).max()
    return rel, mx


def assert_parity(got, ref, what=""):
    rel, mx = errors(got, ref)
    assert np.isfinite(rel) and rel <= REL_L2_TOL, f"{what}: rel L2 {rel:.3e} > {REL_L2_TOL}"
    assert mx <= MAX_ABS_TOL, f"{what}: max abs / max|grid| {mx:.3e} > {MAX_ABS_TOL}"
    return rel, mx
