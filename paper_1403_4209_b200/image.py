"""Headless dirty imager over the C ABI: build_wkernels -> grid -> finalize, on one synthetic configuration or on arrays
from an .npz file (keys uvw_m [nrow,3] f64 metres, baseline [nrow] i32, freqs_hz [nchan] f64, vis [nrow,nchan,npol] c64,
weights [nrow,nchan,npol] f32). Writes the dirty image(s) [npol][N][N] float32 as .npy (the thesis writes FITS, :1680-1687;
no FITS library is assumed here).

    python -m paper_1403_4209_b200.image --config 2 --stokes --out dirty.npy
    python -m paper_1403_4209_b200.image --npz data.npz --grid 2048 --cell-arcsec 14.57 --wplanes 64 --max-support 65 --out dirty.npy
"""
from __future__ import annotations

import argparse
import math

import numpy as np


def main():
    import torch
    from . import build, synth
    from .binding import Gridder
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=0, help="BASELINE.json configuration 1..5")
    ap.add_argument("--npz")
    ap.add_argument("--grid", type=int, default=1024)
    ap.add_argument("--cell-arcsec", type=float, default=10.0)
    ap.add_argument("--wplanes", type=int, default=1)
    ap.add_argument("--oversampling", type=int, default=8)
    ap.add_argument("--max-support", type=int, default=33)
    ap.add_argument("--stokes", action="store_true", help="write Stokes I,Q,U,V images (Alg 4.6 step 2) instead of the polarisations")
    ap.add_argument("--out", default="dirty.npy")
    a = ap.parse_args()
    build.build()
    if a.config:
        cfg = synth.CONFIGS[a.config - 1]
        wl = synth.make_workload(cfg)
        n, cell, P, beta, sup, w_max = cfg.grid_n, wl["cell_rad"], cfg.n_wplanes, cfg.oversampling, wl["supports"], wl["w_max"]
    elif a.npz:
        d = np.load(a.npz)
        wl = dict(uvw_m=np.ascontiguousarray(d["uvw_m"], dtype=np.float64), baseline=np.ascontiguousarray(d["baseline"], dtype=np.int32),
                  freqs_hz=np.ascontiguousarray(d["freqs_hz"], dtype=np.float64), vis=np.ascontiguousarray(d["vis"], dtype=np.complex64),
                  weights=np.ascontiguousarray(d["weights"], dtype=np.float32))
        n, cell, P, beta = a.grid, math.radians(a.cell_arcsec / 3600.0), a.wplanes, a.oversampling
        sup = None                                       # automatic supports (1e-3 rule)
        w_max = float(np.abs(wl["uvw_m"][:, 2]).max() * wl["freqs_hz"].max() / synth.C_M_S)
    else:
        ap.error("give --config or --npz")
    npol = wl["vis"].shape[2]
    max_support = int(sup.max()) if sup is not None else a.max_support
    g = Gridder(n, cell, P, beta, max_support, npol)
    g.allocate(sup)
    g.build_wkernels(w_max if P > 1 else 0.0)
    g.grid_visibilities_host(wl["uvw_m"], wl["baseline"], wl["freqs_hz"], np.ascontiguousarray(wl["vis"]), wl["weights"])
    g.set_stokes_output(a.stokes)
    img, norm = g.finalize()
    gridded, dropped, updates = g.stats()
    np.save(a.out, img.cpu().numpy())
    print(f"{a.out}: {npol} x {n} x {n}; supports {int(g.supports.min())}..{int(g.supports.max())}; "
          f"{gridded} records gridded, {dropped} dropped, {updates} grid-point updates; normaliser {norm}")
    del torch


if __name__ == "__main__":
    main()
