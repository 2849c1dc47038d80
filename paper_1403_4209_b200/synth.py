"""Seeded synthetic interferometer workloads (inputs only; no gridding arithmetic).

Stand-ins for the thesis's LOFAR data sets (Table 5.2), which
are not available. The five configurations restate BASELINE.json `configs`;
the recipe (station layout, Earth-rotation uvw, cell rule, support law) is the
one in DESIGN.md "Input recipe". This module serves
BOTH the oracle tests and the CUDA path as *data*; it contains none of the
method's arithmetic (no index computation, no kernels, no gridding).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

C_M_S = 299792458.0
SEED0 = 14034209
LAT_DEG = 52.91


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    grid_n: int
    n_pol: int
    n_chan: int
    f0_hz: float
    f1_hz: float
    n_station: int
    r_core_m: float      # uniform-disk radius (core)
    r_max_m: float       # outer radius of the log-radial part (== r_core_m: disk only)
    core_frac: float
    n_time: int
    ha0_h: float
    ha1_h: float
    dec_deg: float
    n_wplanes: int
    s_min: int
    s_max: int
    oversampling: int
    weights: str         # "one" | "uniform" | "lognormal"


CONFIGS = [
    Config("cfg1_tiny_plain", 256, 1, 1, 150e6, 150e6, 8, 2e3, 2e3, 1.0, 64, -1, 1, 45.0, 1, 7, 7, 8, "one"),
    Config("cfg2_small_wproj", 1024, 4, 16, 120e6, 180e6, 64, 10e3, 10e3, 1.0, 256, -3, 3, 30.0, 32, 7, 33, 8, "uniform"),
    Config("cfg3_medium", 4096, 4, 64, 110e6, 190e6, 128, 2e3, 50e3, 0.7, 512, -4, 4, 60.0, 128, 9, 65, 8, "uniform"),
    Config("cfg4_large", 8192, 4, 32, 50e6, 250e6, 256, 2e3, 100e3, 0.7, 256, -6, 6, 10.0, 256, 9, 129, 8, "uniform"),
    Config("cfg5_stress", 16384, 4, 16, 100e6, 200e6, 512, 5e3, 150e3, 0.7, 128, -2, 2, -30.0, 512, 9, 129, 8, "lognormal"),
]


def support_table(n_wplanes: int, s_min: int, s_max: int, law: str = "w") -> np.ndarray:
    """Prescribed odd support per w-plane (reading 8): linear in |w|
    (law="w", planes are spaced in sqrt(w) so this is quadratic in p) or linear
    in the plane index (law="k")."""
    if n_wplanes == 1:
        return np.array([s_min], dtype=np.int32)
    p = np.arange(n_wplanes, dtype=np.float64) / (n_wplanes - 1)
    frac = p * p if law == "w" else p
    return (s_min + 2 * np.floor((s_max - s_min) / 2 * frac + 0.5)).astype(np.int32)


def _stations(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    n = cfg.n_station
    n_core = n if cfg.r_max_m <= cfg.r_core_m else int(round(cfg.core_frac * n))
    r = np.empty(n)
    r[:n_core] = cfg.r_core_m * np.sqrt(rng.random(n_core))
    if n_core < n:
        r[n_core:] = cfg.r_core_m * (cfg.r_max_m / cfg.r_core_m) ** rng.random(n - n_core)
    az = 2 * math.pi * rng.random(n)
    return np.stack([r * np.cos(az), r * np.sin(az)], axis=1)  # (E, N) metres


def make_rows(cfg: Config, seed: int | None = None):
    """uvw in metres [nrow][3] (time-major, all baselines per time step, like a
    MeasurementSet) and baseline ids [nrow]."""
    idx = CONFIGS.index(cfg) if cfg in CONFIGS else 0
    rng = np.random.Generator(np.random.Philox(SEED0 + idx if seed is None else seed))
    en = _stations(cfg, rng)
    i, j = np.triu_indices(cfg.n_station, 1)
    d_e = en[j, 0] - en[i, 0]
    d_n = en[j, 1] - en[i, 1]
    lat = math.radians(LAT_DEG)
    lx, ly, lz = -math.sin(lat) * d_n, d_e, math.cos(lat) * d_n
    ha = np.radians(np.linspace(cfg.ha0_h, cfg.ha1_h, cfg.n_time) * 15.0)[:, None]
    dec = math.radians(cfg.dec_deg)
    sh, ch, sd, cd = np.sin(ha), np.cos(ha), math.sin(dec), math.cos(dec)
    u = sh * lx + ch * ly
    v = -sd * ch * lx + sd * sh * ly + cd * lz
    w = cd * ch * lx - cd * sh * ly + sd * lz
    uvw = np.stack([u, v, w], axis=-1).reshape(-1, 3).astype(np.float64)
    n_bl = i.size
    baseline = np.tile(np.arange(n_bl, dtype=np.int32), cfg.n_time)
    return np.ascontiguousarray(uvw), baseline, rng


def make_workload(cfg: Config, support_law: str = "w", with_vis: bool = True,
                  max_rows: int | None = None):
    """Full input set for one configuration. `max_rows` keeps only the first
    rows (whole time steps first) - used for bounded CPU samples."""
    uvw, baseline, rng = make_rows(cfg)
    freqs = np.linspace(cfg.f0_hz, cfg.f1_hz, cfg.n_chan).astype(np.float64)
    f_top = float(freqs.max())
    uv_max = float(np.abs(uvw[:, :2]).max()) * f_top / C_M_S
    du = uv_max / (0.4 * cfg.grid_n)                  # uv cell, wavelengths
    cell_rad = 1.0 / (cfg.grid_n * du)
    w_max = float(np.abs(uvw[:, 2]).max()) * f_top / C_M_S
    if max_rows is not None:
        uvw, baseline = uvw[:max_rows], baseline[:max_rows]
    out = dict(cfg=cfg, uvw_m=uvw, baseline=baseline, freqs_hz=freqs, cell_rad=cell_rad,
               du=du, w_max=w_max,
               supports=support_table(cfg.n_wplanes, cfg.s_min, cfg.s_max, support_law))
    if with_vis:
        shape = (uvw.shape[0], cfg.n_chan, cfg.n_pol)
        vis = np.empty(shape + (2,), dtype=np.float32)
        step = max(1, (1 << 24) // (cfg.n_chan * cfg.n_pol * 2))
        for s in range(0, shape[0], step):             # bounded temporaries
            vis[s:s + step] = rng.standard_normal(vis[s:s + step].shape, dtype=np.float32)
        if cfg.weights == "one":
            wt = np.ones(shape, dtype=np.float32)
        elif cfg.weights == "uniform":
            wt = (0.5 + 0.5 * rng.random(shape, dtype=np.float32)).astype(np.float32)
        else:
            wt = np.exp(0.5 * rng.standard_normal(shape, dtype=np.float32)).astype(np.float32)
        out["vis"] = vis.view(np.complex64)[..., 0]
        out["weights"] = wt
    return out
