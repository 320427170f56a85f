"""TEST INFRASTRUCTURE -- float64 CPU oracle (ctypes wrapper around oracle/gridder_oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  The product (paper_1605_07023_b200) never does and has no CPU fallback.

What it computes and which passage each step follows is documented in gridder_oracle.cpp; the
readings of the paper are DESIGN.md R1-R24.  "Parity unpinned": physical tap positions inside the
table (see gridder_oracle.cpp header).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gridder_oracle.cpp")
_LIB = os.path.join(_HERE, "libgridder_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O3 -fopenmp (no CUDA headers, separate translation unit)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O3", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c_int, c_ll, vp = ctypes.c_int, ctypes.c_longlong, ctypes.c_void_p
        lib.oracle_quantise.argtypes = [c_int] * 4 + [c_ll] + [vp] * 7
        lib.oracle_quantise.restype = c_int
        lib.oracle_grid.argtypes = [c_int] * 5 + [c_ll] + [vp] * 5 + [c_int] * 3 + [vp]
        lib.oracle_grid.restype = c_int
        lib.oracle_degrid.argtypes = [c_int] * 5 + [c_ll] + [vp] * 5
        lib.oracle_grid_dense.argtypes = [c_int] * 5 + [c_ll] + [vp] * 5
        lib.oracle_grid_dense_pol.argtypes = [c_int] * 5 + [c_ll] + [vp] * 5
        lib.oracle_degrid.restype = c_int
        lib.oracle_max_threads.restype = c_int
        _lib = lib
    return _lib


def _f32(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def _c64(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.complex64, a.dtype
    return a


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def quantise(grid_size, support, oversample, n_wplanes, uvw):
    """Q and W of DESIGN.md R4/R5 -> dict of int32 arrays i0, j0, su, sv, wp and uint8 valid."""
    lib = _load()
    uvw = _f32(uvw)
    n = uvw.shape[0]
    out = {k: np.empty(n, dtype=np.int32) for k in ("i0", "j0", "su", "sv", "wp")}
    out["valid"] = np.empty(n, dtype=np.uint8)
    rc = lib.oracle_quantise(grid_size, support, oversample, n_wplanes, n, uvw.ctypes.data,
                             *(out[k].ctypes.data for k in ("i0", "j0", "su", "sv", "wp", "valid")))
    if rc != 0:
        raise ValueError("oracle_quantise: invalid arguments")
    return out


def grid(grid_size, support, oversample, n_wplanes, n_pol, uvw, vis, weights, kernel,
         rows=None, n_threads=0, out=None, return_valid=False):
    """complex128 grid [rows][N][P] (+= into ``out`` if given).  rows=(lo, hi) restricts to a row band."""
    lib = _load()
    uvw = _f32(uvw)
    n = uvw.shape[0]
    vis = _c64(vis).reshape(n, n_pol)
    weights = _f32(weights, (n,))
    kernel = _c64(kernel)
    assert kernel.shape == (n_wplanes, oversample, support), kernel.shape
    lo, hi = (0, grid_size) if rows is None else rows
    if out is None:
        out = np.zeros((hi - lo, grid_size, n_pol), dtype=np.complex128)
    assert out.shape == (hi - lo, grid_size, n_pol) and out.dtype == np.complex128
    assert out.flags.c_contiguous
    nv = ctypes.c_longlong(0)
    rc = lib.oracle_grid(grid_size, support, oversample, n_wplanes, n_pol, n, uvw.ctypes.data,
                         vis.ctypes.data, weights.ctypes.data, kernel.ctypes.data, out.ctypes.data,
                         lo, hi, n_threads, ctypes.addressof(nv))
    if rc != 0:
        raise ValueError("oracle_grid: invalid arguments")
    return (out, int(nv.value)) if return_valid else out


def grid_dense(grid_size, support, oversample, n_wplanes, n_pol, uvw, vis, weights, kernel2d):
    """Gridding with a dense (non-separable) GCF table kernel2d[wp][sv][su][tj][ti] (SURVEY NEXT-4,
    PAPER.md:97, 186): complex128 grid [N][N][P].  Serial; small cases only."""
    lib = _load()
    uvw = _f32(uvw)
    n = uvw.shape[0]
    vis = _c64(vis).reshape(n, n_pol)
    weights = _f32(weights, (n,))
    kernel2d = _c64(kernel2d)
    assert kernel2d.shape == (n_wplanes, oversample, oversample, support, support), kernel2d.shape
    out = np.zeros((grid_size, grid_size, n_pol), dtype=np.complex128)
    rc = lib.oracle_grid_dense(grid_size, support, oversample, n_wplanes, n_pol, n, uvw.ctypes.data,
                               vis.ctypes.data, weights.ctypes.data, kernel2d.ctypes.data, out.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_grid_dense: invalid arguments")
    return out


def grid_dense_pol(grid_size, support, oversample, n_wplanes, n_pol, uvw, vis, weights, kernel2d):
    """Gridding with one dense GCF table per polarisation, kernel2d[p][wp][sv][su][tj][ti] (SURVEY NEXT-4,
    PAPER.md:97, 186): complex128 grid [N][N][P].  Serial; small cases only."""
    lib = _load()
    uvw = _f32(uvw)
    n = uvw.shape[0]
    vis = _c64(vis).reshape(n, n_pol)
    weights = _f32(weights, (n,))
    kernel2d = _c64(kernel2d)
    assert kernel2d.shape == (n_pol, n_wplanes, oversample, oversample, support, support), kernel2d.shape
    out = np.zeros((grid_size, grid_size, n_pol), dtype=np.complex128)
    rc = lib.oracle_grid_dense_pol(grid_size, support, oversample, n_wplanes, n_pol, n, uvw.ctypes.data,
                                   vis.ctypes.data, weights.ctypes.data, kernel2d.ctypes.data, out.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_grid_dense_pol: invalid arguments")
    return out


def degrid(grid_size, support, oversample, n_wplanes, n_pol, uvw, weights, kernel, grid_in):
    """Adjoint of grid() (pin P7 only): complex128 [n_vis][P]."""
    lib = _load()
    uvw = _f32(uvw)
    n = uvw.shape[0]
    weights = _f32(weights, (n,))
    kernel = _c64(kernel)
    g = np.ascontiguousarray(grid_in, dtype=np.complex128)
    assert g.shape == (grid_size, grid_size, n_pol)
    out = np.empty((n, n_pol), dtype=np.complex128)
    rc = lib.oracle_degrid(grid_size, support, oversample, n_wplanes, n_pol, n, uvw.ctypes.data,
                           weights.ctypes.data, kernel.ctypes.data, g.ctypes.data, out.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_degrid: invalid arguments")
    return out


def compress(grid_size, support, oversample, n_wplanes, uvw, vis, weights):
    """Compression as the paper describes it ("merge adjacent visibilities with identical
    oversampled position"; a compressed sample carries integer grid coordinates, sub-grid
    coordinates, w-plane index and pre-weighted values).  Walks the samples in input order; a run is a
    maximal sequence of CONSECUTIVE valid samples with equal (i0, su, j0, sv, wp); skipped samples (R7)
    end a run and produce nothing.  Returns (heads int64 [n_c] = index of each run's first sample,
    merged complex128 [n_c][P] = sum over the run of weight * vis in float64, input order).
    Test infrastructure only, like everything in oracle/."""
    q = quantise(grid_size, support, oversample, n_wplanes, uvw)
    v = np.asarray(vis).reshape(len(q["valid"]), -1)
    w = np.asarray(weights, dtype=np.float64)
    heads, merged = [], []
    prev = None
    for n in range(len(w)):                           # plain loop: small cases only
        if not q["valid"][n]:
            prev = None
            continue
        key = (int(q["i0"][n]), int(q["su"][n]), int(q["j0"][n]), int(q["sv"][n]), int(q["wp"][n]))
        term = w[n] * v[n].astype(np.complex128)
        if key == prev:
            merged[-1] = merged[-1] + term
        else:
            heads.append(n)
            merged.append(term)
            prev = key
    P = v.shape[1]
    return np.asarray(heads, dtype=np.int64), np.asarray(merged, dtype=np.complex128).reshape(len(heads), P)
