"""Thin ctypes binding over libgridb200.so (include/grid.h).  Argument marshalling only: every step
of the hot path runs in the library's CUDA kernels.  torch is used for device memory and streams.

There is no CPU fallback: if the shared library is missing, importing this module raises.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# GRIDB200_LIB: another build of the same library (the bounds-checked one of tests/test_gpu_checked_build.py)
LIB_PATH = os.environ.get("GRIDB200_LIB") or os.path.join(_HERE, "libgridb200.so")

GRID_OK, GRID_ERR_INVALID_ARG, GRID_ERR_UNSUPPORTED, GRID_ERR_CUDA, GRID_ERR_STATE = 0, -1, -2, -3, -4

EXPORTS = (
    "grid_plan_create", "grid_plan_set_samples", "grid_plan_set_layout", "grid_plan_workspace_bytes",
    "grid_plan_set_workspace", "grid_execute", "grid_execute_static", "grid_compress", "grid_execute_compressed", "grid_execute_dense", "grid_execute_dense_pol", "grid_degrid", "grid_plan_set_degrid_gather", "grid_quantise", "grid_plan_set_tuning",
    "grid_plan_get_info", "grid_plan_set_traversal", "grid_plan_set_kernel_events", "grid_plan_set_chunk_order", "grid_plan_set_sample_order", "grid_plan_set_pol_split", "grid_plan_autotune", "grid_plan_autotune_candidates", "grid_plan_last_launches", "grid_plan_debug_counters", "grid_plan_destroy", "grid_last_error",
)

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
        "(nvcc, sm_100a).  The gridder has no CPU fallback.")

_lib = ctypes.CDLL(LIB_PATH)
_vp, _int, _ll, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong, ctypes.c_size_t
_lib.grid_plan_create.argtypes = [_int] * 5
_lib.grid_plan_create.restype = _vp
_lib.grid_plan_set_samples.argtypes = [_vp, _ll]
_lib.grid_plan_set_layout.argtypes = [_vp, _int, _int, _int]
_lib.grid_plan_workspace_bytes.argtypes = [_vp]
_lib.grid_plan_workspace_bytes.restype = _sz
_lib.grid_plan_set_workspace.argtypes = [_vp, _vp, _sz]
_lib.grid_execute.argtypes = [_vp] * 7
_lib.grid_execute_static.argtypes = [_vp] * 7
_lib.grid_quantise.argtypes = [_vp, _vp, _ll, _vp, _vp]
_lib.grid_compress.argtypes = [_vp] * 8
_lib.grid_execute_dense.argtypes = [_vp] * 7
_lib.grid_execute_dense_pol.argtypes = [_vp] * 7
_lib.grid_degrid.argtypes = [_vp] * 7
_lib.grid_plan_set_degrid_gather.argtypes = [_vp, _int]
_lib.grid_execute_compressed.argtypes = [_vp, _vp, _vp, _ll, _vp, _vp, _vp]
_lib.grid_plan_set_tuning.argtypes = [_vp] + [_int] * 7
_lib.grid_plan_get_info.argtypes = [_vp, _vp]
_lib.grid_plan_set_traversal.argtypes = [_vp, _int, _int]
_lib.grid_plan_set_kernel_events.argtypes = [_vp, _vp, _vp]
_lib.grid_plan_set_chunk_order.argtypes = [_vp, _int]
_lib.grid_plan_set_sample_order.argtypes = [_vp, _int]
_lib.grid_plan_set_pol_split.argtypes = [_vp, _int]
_lib.grid_plan_autotune_candidates.argtypes = [_vp, _vp, _int]
_lib.grid_plan_autotune.argtypes = [_vp, _ll, ctypes.c_uint, _vp, _int, _vp]
_lib.grid_plan_last_launches.argtypes = [_vp]
_lib.grid_plan_debug_counters.argtypes = [_vp, _vp, _vp]
_lib.grid_plan_destroy.argtypes = [_vp]
_lib.grid_plan_destroy.restype = None
_lib.grid_last_error.restype = ctypes.c_char_p


class GridError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: error {code}: {_lib.grid_last_error().decode()}")


def grid_last_error() -> str:
    return _lib.grid_last_error().decode()


def _check(rc: int, where: str) -> None:
    if rc != GRID_OK:
        raise GridError(rc, where)


def _ptr(t, dtype, what):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{what}: expected a CUDA torch.Tensor (device pointers only; no CPU fallback)")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{what}: expected contiguous {dtype}, got {t.dtype} contiguous={t.is_contiguous()}")
    return t.data_ptr()


def _stream(stream):
    import torch
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


INFO_FIELDS = ("variant", "cu", "cv", "bin_u", "bin_v", "team_threads", "teams_per_cta",
               "threads_per_cta", "batch", "chunk", "ctas_per_sm", "smem_bytes", "n_sm", "traversal", "time_block", "chunk_order", "pol_split", "groups_per_cta", "taps_global", "sample_order")


class GridPlan:
    """Owns a grid_plan* (same names as the C ABI: set_samples, set_layout, set_workspace, execute)."""

    def __init__(self, grid_size, support, oversample, n_wplanes, n_pol):
        self._h = _lib.grid_plan_create(grid_size, support, oversample, n_wplanes, n_pol)
        if not self._h:
            raise GridError(GRID_ERR_INVALID_ARG, "grid_plan_create")
        self.grid_size, self.support, self.oversample = grid_size, support, oversample
        self.n_wplanes, self.n_pol = n_wplanes, n_pol
        self.n_vis = None
        self._workspace = None

    def destroy(self):
        if getattr(self, "_h", None):
            _lib.grid_plan_destroy(self._h)
            self._h = None
            self._workspace = None

    __del__ = destroy

    def set_samples(self, n_vis: int):
        _check(_lib.grid_plan_set_samples(self._h, n_vis), "grid_plan_set_samples")
        self.n_vis = n_vis

    def set_layout(self, n_baselines: int, n_times: int, n_channels: int):
        _check(_lib.grid_plan_set_layout(self._h, n_baselines, n_times, n_channels), "grid_plan_set_layout")

    def workspace_bytes(self) -> int:
        return int(_lib.grid_plan_workspace_bytes(self._h))

    def set_workspace(self, tensor):
        import torch
        ptr = _ptr(tensor, torch.uint8, "workspace")
        _check(_lib.grid_plan_set_workspace(self._h, ptr, tensor.numel()), "grid_plan_set_workspace")
        self._workspace = tensor          # keep the caller's buffer alive

    def allocate_workspace(self, device="cuda"):
        import torch
        self.set_workspace(torch.empty(max(self.workspace_bytes(), 256), dtype=torch.uint8, device=device))

    def set_tuning(self, variant=-1, cu=0, cv=0, threads_per_cta=0, batch=0, chunk=0, ctas_per_sm=0):
        _check(_lib.grid_plan_set_tuning(self._h, variant, cu, cv, threads_per_cta, batch, chunk, ctas_per_sm),
               "grid_plan_set_tuning")

    def set_traversal(self, mode=-1, time_block=0):
        _check(_lib.grid_plan_set_traversal(self._h, mode, time_block), "grid_plan_set_traversal")

    def set_pol_split(self, lanes=1):
        _check(_lib.grid_plan_set_pol_split(self._h, lanes), "grid_plan_set_pol_split")

    def set_chunk_order(self, mode=-1):
        _check(_lib.grid_plan_set_chunk_order(self._h, mode), "grid_plan_set_chunk_order")

    def set_sample_order(self, mode=-1):
        _check(_lib.grid_plan_set_sample_order(self._h, mode), "grid_plan_set_sample_order")

    def autotune_candidates(self):
        """grid_plan_autotune_candidates: list of (cu, cv, pol_split) blocks that fit this plan, the current one first."""
        out = (ctypes.c_int * (3 * 32))()
        n = _lib.grid_plan_autotune_candidates(self._h, out, 32)
        if n < 0:
            raise GridError(n, "grid_plan_autotune_candidates")
        return [(out[3 * k], out[3 * k + 1], out[3 * k + 2]) for k in range(n)]

    def autotune(self, n_samples=0, seed=1, stream=None):
        """grid_plan_autotune: times every candidate on a synthetic data set, installs the fastest.
        Returns [((cu, cv, pol_split), microseconds), ...] in candidate order."""
        cands = self.autotune_candidates()
        res = (ctypes.c_float * 32)()
        _check(_lib.grid_plan_autotune(self._h, n_samples, seed, res, 32, _stream(stream)), "grid_plan_autotune")
        return [(c, float(res[k])) for k, c in enumerate(cands)]

    def info(self) -> dict:
        out = (ctypes.c_int * 20)()
        _check(_lib.grid_plan_get_info(self._h, out), "grid_plan_get_info")
        return dict(zip(INFO_FIELDS, list(out)))

    def set_kernel_events(self, ev_start=None, ev_stop=None):
        """torch.cuda.Event pair (enable_timing=True, already created) recorded around the gridding kernel."""
        a = ev_start.cuda_event if ev_start is not None else None
        b = ev_stop.cuda_event if ev_stop is not None else None
        _check(_lib.grid_plan_set_kernel_events(self._h, a, b), "grid_plan_set_kernel_events")

    def debug_counters(self, stream=None):
        """grid_plan_debug_counters: bounds violations counted by a -DGRIDB200_CHECK build (zeros otherwise)."""
        out = (ctypes.c_uint * 8)()
        _check(_lib.grid_plan_debug_counters(self._h, out, _stream(stream)), "grid_plan_debug_counters")
        return list(out)

    def last_launches(self) -> int:
        return int(_lib.grid_plan_last_launches(self._h))

    def _check_samples(self, uvw=None, vis=None, weights=None, grid=None, vis_out=None):
        """Sizes against the plan (every wrapper: an undersized array would be read or written out of bounds on the
        device).  Marshalling only -- no arithmetic on the data."""
        n = self.n_vis
        if n is None:
            _lib.grid_plan_set_samples(self._h, -1)            # leaves "invalid argument" in grid_last_error
            raise GridError(GRID_ERR_STATE, "set_samples has not been called")
        if uvw is not None and uvw.numel() != 3 * n:
            raise ValueError(f"uvw must hold [n_vis = {n}][3] floats, got {uvw.numel()} elements")
        if vis is not None and vis.numel() != n * self.n_pol:
            raise ValueError(f"vis must hold [n_vis = {n}][n_pol = {self.n_pol}] complex values, got {vis.numel()}")
        if weights is not None and weights.numel() != n:
            raise ValueError(f"weights must hold n_vis = {n} floats, got {weights.numel()}")
        if vis_out is not None and vis_out.numel() != n * self.n_pol:
            raise ValueError(f"vis_out must hold [n_vis = {n}][n_pol = {self.n_pol}] complex values, got {vis_out.numel()}")
        if grid is not None and grid.numel() != self.grid_size * self.grid_size * self.n_pol:
            raise ValueError("grid must be [N][N][n_pol]")

    def execute(self, uvw, vis, weights, conv_kernel, grid, stream=None):
        """grid += gridded samples (grid_execute).  All arguments are CUDA tensors:
        uvw float32 [n][3], vis complex64 [n][P], weights float32 [n],
        conv_kernel complex64 [W][O][S], grid complex64 [N][N][P]."""
        import torch
        self._check_samples(uvw, vis, weights, grid)
        if conv_kernel.numel() != self.n_wplanes * self.oversample * self.support:
            raise ValueError("conv_kernel must be [n_wplanes][oversample][support]")
        rc = _lib.grid_execute(self._h, _ptr(uvw, torch.float32, "uvw"), _ptr(vis, torch.complex64, "vis"),
                               _ptr(weights, torch.float32, "weights"),
                               _ptr(conv_kernel, torch.complex64, "conv_kernel"),
                               _ptr(grid, torch.complex64, "grid"), _stream(stream))
        _check(rc, "grid_execute")

    def execute_static(self, uvw, vis, weights, conv_kernel, grid, stream=None):
        """grid_execute_static: grid_execute with the workspace in the library's static device array -- no allocation;
        at most GRID_STATIC_SCRATCH_BYTES (20 MiB, about 1.2 million samples) per call; calls must not overlap on the GPU."""
        import torch
        self._check_samples(uvw, vis, weights, grid)
        if conv_kernel.numel() != self.n_wplanes * self.oversample * self.support:
            raise ValueError("conv_kernel must be [n_wplanes][oversample][support]")
        rc = _lib.grid_execute_static(self._h, _ptr(uvw, torch.float32, "uvw"), _ptr(vis, torch.complex64, "vis"),
                                      _ptr(weights, torch.float32, "weights"),
                                      _ptr(conv_kernel, torch.complex64, "conv_kernel"),
                                      _ptr(grid, torch.complex64, "grid"), _stream(stream))
        _check(rc, "grid_execute_static")

    def execute_dense(self, uvw, vis, weights, conv_kernel_2d, grid, stream=None):
        """grid_execute_dense: conv_kernel_2d complex64 [W][O][O][S][S] (plane, sv, su, row, column)."""
        import torch
        self._check_samples(uvw, vis, weights, grid)
        if conv_kernel_2d.numel() != self.n_wplanes * self.oversample ** 2 * self.support ** 2:
            raise ValueError("conv_kernel_2d must be [n_wplanes][oversample][oversample][support][support]")
        rc = _lib.grid_execute_dense(self._h, _ptr(uvw, torch.float32, "uvw"), _ptr(vis, torch.complex64, "vis"),
                                     _ptr(weights, torch.float32, "weights"),
                                     _ptr(conv_kernel_2d, torch.complex64, "conv_kernel_2d"),
                                     _ptr(grid, torch.complex64, "grid"), _stream(stream))
        _check(rc, "grid_execute_dense")

    def execute_dense_pol(self, uvw, vis, weights, conv_kernel_2d_pol, grid, stream=None):
        """grid_execute_dense_pol: conv_kernel_2d_pol complex64 [P][W][O][O][S][S] (one dense table per polarisation)."""
        import torch
        self._check_samples(uvw, vis, weights, grid)
        if conv_kernel_2d_pol.numel() != self.n_pol * self.n_wplanes * self.oversample ** 2 * self.support ** 2:
            raise ValueError("conv_kernel_2d_pol must be [n_pol][n_wplanes][oversample][oversample][support][support]")
        rc = _lib.grid_execute_dense_pol(self._h, _ptr(uvw, torch.float32, "uvw"), _ptr(vis, torch.complex64, "vis"),
                                         _ptr(weights, torch.float32, "weights"),
                                         _ptr(conv_kernel_2d_pol, torch.complex64, "conv_kernel_2d_pol"),
                                         _ptr(grid, torch.complex64, "grid"), _stream(stream))
        _check(rc, "grid_execute_dense_pol")

    def compress(self, uvw, vis, weights, stream=None):
        """grid_compress: returns (records uint8 [n_c][8], vis complex64 [n_c][P], n_c) -- CUDA tensors trimmed
        to the compressed count (one host sync to read it)."""
        import torch
        self._check_samples(uvw, vis, weights)
        n = self.n_vis
        recs = torch.empty((max(n, 1), 8), dtype=torch.uint8, device=uvw.device)
        cvis = torch.empty((max(n, 1), self.n_pol), dtype=torch.complex64, device=uvw.device)
        count = torch.zeros(1, dtype=torch.int64, device=uvw.device)
        rc = _lib.grid_compress(self._h, _ptr(uvw, torch.float32, "uvw"), _ptr(vis, torch.complex64, "vis"),
                                _ptr(weights, torch.float32, "weights"), recs.data_ptr(), cvis.data_ptr(),
                                count.data_ptr(), _stream(stream))
        _check(rc, "grid_compress")
        n_c = int(count.item())
        return recs[:n_c], cvis[:n_c], n_c

    def execute_compressed(self, records, vis, conv_kernel, grid, stream=None):
        """grid_execute_compressed on the output of compress()."""
        import torch
        self._check_samples(grid=grid)
        n_c = records.shape[0]
        if records.numel() != n_c * 8 or vis.numel() != n_c * self.n_pol or n_c > self.n_vis:
            raise ValueError("records must be [n_c][8] bytes and vis [n_c][n_pol] with n_c <= n_vis")
        if conv_kernel.numel() != self.n_wplanes * self.oversample * self.support:
            raise ValueError("conv_kernel must be [n_wplanes][oversample][support]")
        rc = _lib.grid_execute_compressed(self._h, _ptr(records, torch.uint8, "records") if n_c else None,
                                          _ptr(vis, torch.complex64, "vis") if n_c else None, n_c,
                                          _ptr(conv_kernel, torch.complex64, "conv_kernel"),
                                          _ptr(grid, torch.complex64, "grid"), _stream(stream))
        _check(rc, "grid_execute_compressed")

    def set_degrid_gather(self, on=1):
        _check(_lib.grid_plan_set_degrid_gather(self._h, on), "grid_plan_set_degrid_gather")

    def degrid(self, uvw, weights, conv_kernel, grid, vis_out=None, stream=None):
        """grid_degrid: vis_out complex64 [n][P] (allocated if None) = adjoint of execute() applied to grid."""
        import torch
        self._check_samples(uvw, None, weights, grid)
        n = self.n_vis
        if vis_out is None:
            vis_out = torch.empty((n, self.n_pol), dtype=torch.complex64, device=grid.device)
        self._check_samples(vis_out=vis_out)
        if conv_kernel.numel() != self.n_wplanes * self.oversample * self.support:
            raise ValueError("conv_kernel must be [n_wplanes][oversample][support]")
        if n == 0:
            return vis_out
        rc = _lib.grid_degrid(self._h, _ptr(uvw, torch.float32, "uvw"), _ptr(weights, torch.float32, "weights"),
                              _ptr(conv_kernel, torch.complex64, "conv_kernel"), _ptr(grid, torch.complex64, "grid"),
                              _ptr(vis_out, torch.complex64, "vis_out"), _stream(stream))
        _check(rc, "grid_degrid")
        return vis_out

    def quantise(self, uvw, stream=None):
        """Step a1 alone -> int32 CUDA tensor [n][6] = i0, j0, su, sv, wp, valid."""
        import torch
        n = uvw.shape[0]
        out = torch.empty((n, 6), dtype=torch.int32, device=uvw.device)
        _check(_lib.grid_quantise(self._h, _ptr(uvw, torch.float32, "uvw"), n, out.data_ptr(), _stream(stream)),
               "grid_quantise")
        return out


def grid_visibilities(grid_size, support, oversample, n_wplanes, n_pol, uvw, vis, weights, conv_kernel,
                      grid=None, layout=None, tuning=None):
    """One-shot convenience wrapper over the plan calls; returns the (accumulated) grid tensor."""
    import torch
    plan = GridPlan(grid_size, support, oversample, n_wplanes, n_pol)
    try:
        plan.set_samples(uvw.shape[0])
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
        plan.allocate_workspace(uvw.device)
        if grid is None:
            grid = torch.zeros((grid_size, grid_size, n_pol), dtype=torch.complex64, device=uvw.device)
        plan.execute(uvw, vis, weights, conv_kernel, grid)
        torch.cuda.current_stream().synchronize()
    finally:
        plan.destroy()
    return grid
