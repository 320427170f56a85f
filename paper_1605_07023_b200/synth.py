"""Seeded synthetic workloads (inputs only -- none of the gridding arithmetic lives here).

These arrays stand in for the paper's simulated MeerKAT data set (section 5;
URL at PAPER.md:121), which is not available.  Shapes follow BASELINE.json:configs[0..4]; every
choice the configs leave open is listed in DESIGN.md ("Input recipe") and SURVEY.md 8(d).

Both the CUDA path (tests, bench.py) and the float64 oracle are fed from this module; it imports
neither.  All physics is float64 numpy; one final cast to float32.

RNG: ``numpy.random.default_rng(seed)``; draw order: antenna radii, antenna angles, vis re/im,
weights, kernel noise.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Optional

import numpy as np

C_LIGHT = 299792458.0
LATITUDE_DEG = -30.0
DEC_DEG = -30.0


@dataclass(frozen=True)
class Config:
    name: str
    seed: int
    n_ant: int
    layout: str            # "disk" | "logradial"
    radius_m: float
    n_times: int
    hours: float
    n_chan: int
    f0_hz: float
    f1_hz: float
    n_pol: int
    grid_size: int
    support: int
    oversample: int
    n_wplanes: int
    kernel: str            # "kb_noise" (configs 0,1,3) | "kb_chirp" (configs 2,4)
    random_weights: bool

    @property
    def n_baselines(self) -> int:
        return self.n_ant * (self.n_ant - 1) // 2

    @property
    def n_vis(self) -> int:
        return self.n_baselines * self.n_times * self.n_chan


CONFIGS = {
    # BASELINE.json:configs[0]
    "cfg0": Config("cfg0", 0, 32, "disk", 2000.0, 32, 1.0, 8, 1.20e9, 1.30e9, 1, 512, 7, 8, 1,
                   "kb_noise", False),
    # BASELINE.json:configs[1]
    "cfg1": Config("cfg1", 1, 64, "disk", 4000.0, 256, 4.0, 64, 0.9e9, 1.7e9, 4, 2048, 8, 8, 1,
                   "kb_noise", True),
    # BASELINE.json:configs[2]
    "cfg2": Config("cfg2", 2, 64, "disk", 8000.0, 128, 6.0, 128, 0.9e9, 1.7e9, 1, 4096, 16, 8, 32,
                   "kb_chirp", False),
    # BASELINE.json:configs[3]
    "cfg3": Config("cfg3", 3, 197, "logradial", 20000.0, 64, 2.0, 64, 0.95e9, 1.76e9, 4, 8192, 8, 8,
                   1, "kb_noise", False),
}


def paper_regime_config(support: int, n_pol: int, n_wplanes: int = 16) -> Config:
    """Shape of the paper's own workload: 64 antennas, one channel, 2 h of 2-s dumps =
    2016 x 3600 = 7 257 600 samples that move a fraction of a cell per dump.  Synthetic antennas and
    visibilities as everywhere else; NOT the paper's data set.  Context measurement only."""
    name = f"paper_S{support}_P{n_pol}" + ("" if n_wplanes == 16 else f"_W{n_wplanes}")
    return Config(name, 7, 64, "disk", 4000.0, 3600, 2.0, 1, 1.4e9, 1.4e9, n_pol, 4096,
                  support, 8, n_wplanes, "kb_chirp", False)


WSTACK_SLICES = 7          # "7 slices"
WSTACK_PLANES = 1229       # "1229 W planes per slice"


def wstack_config(support: int, n_pol: int, n_slices: int = WSTACK_SLICES, planes_per_slice: int = WSTACK_PLANES) -> Config:
    """The paper's W-stacked run (the data is split "into a number of slices by w value", each
    gridded by "a separate kernel-instance" onto its own grid with its own W-projection planes): the paper-shaped
    workload with n_slices * planes_per_slice w-planes; split_wstack() cuts it into the slices."""
    base = paper_regime_config(support, n_pol, n_slices * planes_per_slice)
    return replace(base, name=f"paper_wstack_S{support}_P{n_pol}")


@dataclass
class WSlice:
    index: int
    sample_idx: np.ndarray     # positions of the slice's samples in the full workload (input order kept)
    uvw: np.ndarray            # w relative to the slice's first plane
    vis: np.ndarray
    weights: np.ndarray
    kernel: np.ndarray         # the slice's own planes [planes_per_slice][O][S]


def split_wstack(wl: "Workload", n_slices: int = WSTACK_SLICES):
    """Input preparation of the W-stacked run: slice s takes the samples whose w (in plane units) falls into
    [s, s+1) * planes_per_slice, with w counted from the slice's first plane and the slice's own tap planes."""
    per = wl.cfg.n_wplanes // n_slices
    assert per * n_slices == wl.cfg.n_wplanes
    which = np.minimum((wl.uvw[:, 2] // per).astype(np.int64), n_slices - 1)
    out = []
    for s in range(n_slices):
        idx = np.flatnonzero(which == s)
        uvw = wl.uvw[idx].copy()
        uvw[:, 2] -= np.float32(s * per)                  # exact: an integer taken off a float of larger magnitude
        out.append(WSlice(s, idx, uvw, np.ascontiguousarray(wl.vis[idx]), wl.weights[idx].copy(),
                          np.ascontiguousarray(wl.kernel[s * per:(s + 1) * per])))
    return out


def sweep_config(support: int, n_pol: int) -> Config:
    """BASELINE.json:configs[4]: support/pol sweep on the config-1 array, 4096 grid, 16 chirp planes."""
    base = CONFIGS["cfg1"]
    return replace(base, name=f"cfg4_S{support}_P{n_pol}", n_pol=n_pol, grid_size=4096,
                   support=support, n_wplanes=16, kernel="kb_chirp")


def get_config(name: str) -> Config:
    if name in CONFIGS:
        return CONFIGS[name]
    if name.startswith("paper_wstack_S"):
        sp, p = name[len("paper_wstack_S"):].split("_P")
        return wstack_config(int(sp), int(p))
    if name.startswith("paper_S"):
        s, rest = name[len("paper_S"):].split("_P")
        p, _, w = rest.partition("_W")
        return paper_regime_config(int(s), int(p), int(w) if w else 16)
    if name.startswith("cfg4_S"):
        s, p = name[len("cfg4_S"):].split("_P")
        return sweep_config(int(s), int(p))
    raise KeyError(name)


def shrink(cfg: Config, n_ant: Optional[int] = None, n_times: Optional[int] = None,
           n_chan: Optional[int] = None, grid_size: Optional[int] = None) -> Config:
    """Same recipe, fewer antennas / times / channels (parity cases the oracle finishes in seconds)."""
    return replace(cfg, name=cfg.name + "_small",
                   n_ant=n_ant or cfg.n_ant, n_times=n_times or cfg.n_times,
                   n_chan=n_chan or cfg.n_chan, grid_size=grid_size or cfg.grid_size)


@dataclass
class Workload:
    cfg: Config
    uvw: np.ndarray          # float32 [n_vis][3]  u,v in cells from the centre cell; w in plane units
    vis: np.ndarray          # complex64 [n_vis][P]
    weights: np.ndarray      # float32 [n_vis]
    kernel: np.ndarray       # complex64 [n_wplanes][O][S]


def antenna_positions(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    u1 = rng.random(cfg.n_ant)
    u2 = rng.random(cfg.n_ant)
    if cfg.layout == "disk":
        r = cfg.radius_m * np.sqrt(u1)
    elif cfg.layout == "logradial":
        rmin = cfg.radius_m / 400.0                      # [50 m, 20 km]: median exactly 1 km
        r = rmin * (cfg.radius_m / rmin) ** u1
    else:
        raise ValueError(cfg.layout)
    theta = 2.0 * np.pi * u2
    return np.stack([r * np.cos(theta), r * np.sin(theta), np.zeros_like(r)], axis=1)   # E, N, U


def baseline_uvw_metres(cfg: Config, enu: np.ndarray) -> np.ndarray:
    """[n_baselines][n_times][3] in metres; baselines p<q in triu order."""
    p, q = np.triu_indices(cfg.n_ant, k=1)
    d = enu[q] - enu[p]
    lat = np.deg2rad(LATITUDE_DEG)
    dec = np.deg2rad(DEC_DEG)
    X = -np.sin(lat) * d[:, 1]
    Y = d[:, 0]
    Z = np.cos(lat) * d[:, 1]
    half = 0.5 * cfg.hours * (2.0 * np.pi / 24.0)
    H = np.linspace(-half, half, cfg.n_times)
    sH, cH = np.sin(H)[None, :], np.cos(H)[None, :]
    X, Y, Z = X[:, None], Y[:, None], Z[:, None]
    u = sH * X + cH * Y
    v = -np.sin(dec) * cH * X + np.sin(dec) * sH * Y + np.cos(dec) * Z
    w = np.cos(dec) * cH * X - np.cos(dec) * sH * Y + np.sin(dec) * Z
    return np.stack([u, v, w], axis=2)


def make_uvw(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    enu = antenna_positions(cfg, rng)
    bl = baseline_uvw_metres(cfg, enu)                           # [B][T][3]
    freqs = np.linspace(cfg.f0_hz, cfg.f1_hz, cfg.n_chan)
    scale = freqs / C_LIGHT                                      # metres -> wavelengths
    uv_max = np.sqrt(bl[..., 0] ** 2 + bl[..., 1] ** 2).max() * scale.max()
    w_max = np.abs(bl[..., 2]).max() * scale.max()
    cell = 0.45 * cfg.grid_size / uv_max
    out = np.empty((cfg.n_baselines, cfg.n_times, cfg.n_chan, 3), dtype=np.float32)
    out[..., 0] = bl[:, :, None, 0] * (scale * cell)[None, None, :]
    out[..., 1] = bl[:, :, None, 1] * (scale * cell)[None, None, :]
    wscale = (cfg.n_wplanes / w_max) if w_max > 0 else 0.0
    out[..., 2] = np.abs(bl[:, :, None, 2]) * (scale * wscale)[None, None, :]
    return out.reshape(-1, 3)


def kaiser_bessel(d: np.ndarray, support: int) -> np.ndarray:
    beta = 2.34 * support
    x = 2.0 * d / support
    inside = np.abs(x) <= 1.0
    arg = np.sqrt(np.where(inside, 1.0 - x * x, 0.0))
    return np.where(inside, np.i0(beta * arg) / np.i0(beta), 0.0)


def make_kernel(cfg: Config, rng: Optional[np.random.Generator]) -> np.ndarray:
    """Separable taps k[wp][su][t]; tap t of row su sits at distance d = t - S/2 + 1 - su/O."""
    S, O, W = cfg.support, cfg.oversample, cfg.n_wplanes
    t = np.arange(S, dtype=np.float64)[None, :]
    su = np.arange(O, dtype=np.float64)[:, None]
    d = t - S / 2.0 + 1.0 - su / O                                # [O][S]
    kb = kaiser_bessel(d, S)
    k = np.empty((W, O, S), dtype=np.complex128)
    if cfg.kernel == "kb_noise":
        for wp in range(W):
            k[wp] = kb
        k = k + 1j * rng.normal(0.0, 1e-3, size=k.shape)
    elif cfg.kernel == "kb_chirp":
        for wp in range(W):
            phi = (-2.0 + 4.0 * wp / (W - 1)) if W > 1 else 0.0
            k[wp] = kb * np.exp(2j * np.pi * phi * d * d / (S * S))
    else:
        raise ValueError(cfg.kernel)
    return k.astype(np.complex64)


def make_workload(cfg: Config) -> Workload:
    rng = np.random.default_rng(cfg.seed)
    uvw = make_uvw(cfg, rng)
    n = uvw.shape[0]
    vis = rng.standard_normal((n, cfg.n_pol, 2), dtype=np.float32).view(np.complex64)[..., 0]
    if cfg.random_weights:
        weights = rng.uniform(0.5, 1.0, n).astype(np.float32)
    else:
        weights = np.ones(n, dtype=np.float32)
    kernel = make_kernel(cfg, rng)
    return Workload(cfg, uvw, np.ascontiguousarray(vis), weights, kernel)


def random_problem(seed: int, n_vis: int, grid_size: int, support: int, oversample: int,
                   n_wplanes: int, n_pol: int, spread: float = 0.45, walk: float = 0.0):
    """Unstructured random inputs for property tests (uniform positions or a random walk)."""
    rng = np.random.default_rng(seed)
    if walk > 0.0:
        steps = rng.normal(0.0, walk, size=(n_vis, 2))
        uv = np.cumsum(steps, axis=0)
        uv = (uv + spread * grid_size) % (2 * spread * grid_size) - spread * grid_size
    else:
        uv = rng.uniform(-spread * grid_size, spread * grid_size, size=(n_vis, 2))
    w = rng.uniform(0.0, n_wplanes, size=(n_vis, 1))
    uvw = np.concatenate([uv, w], axis=1).astype(np.float32)
    vis = rng.standard_normal((n_vis, n_pol, 2), dtype=np.float32).view(np.complex64)[..., 0]
    weights = rng.uniform(0.5, 1.0, n_vis).astype(np.float32)
    kernel = (rng.standard_normal((n_wplanes, oversample, support))
              + 1j * rng.standard_normal((n_wplanes, oversample, support))).astype(np.complex64)
    return uvw, np.ascontiguousarray(vis), weights, kernel
