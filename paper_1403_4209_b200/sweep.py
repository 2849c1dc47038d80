"""Fixed-support sweep ("normal" mode of the thesis): a single w=0 kernel trimmed /
padded to support S, swept over S, oversampling and polarisation count on the array of one BASELINE.json
configuration. Reproduces the SHAPE of thesis batches 2-4 (rate against support, :1819-1907); the thesis's ~50 G
updates/s on a GTX 680 (:1986) is context, not a target. Prints one JSON line per point.

    python -m paper_1403_4209_b200.sweep [--config 2] [--supports 7,15,23,31,63,127,255,349,511] [--betas 2,4,8] [--pols 1,2,4]

A point whose pass would exceed --max-updates complex updates is run on the first whole time steps of the array only
(rows are time-major); the JSON line says how many.
"""
from __future__ import annotations

import argparse
import dataclasses
import json

import numpy as np


def main():
    import torch
    from . import build, synth
    from .binding import Gridder
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--supports", default="7,15,23,31,63,127")
    ap.add_argument("--betas", default="8")
    ap.add_argument("--pols", default="4")
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--max-updates", type=float, default=6e12, help="largest pass, in complex updates (time steps are dropped beyond)")
    ap.add_argument("--gather-min-support", type=int, default=None)
    a = ap.parse_args()
    build.build()
    base = synth.CONFIGS[a.config - 1]
    dev = "cuda:0"
    for npol in [int(x) for x in a.pols.split(",")]:
        for beta in [int(x) for x in a.betas.split(",")]:
            cfg = dataclasses.replace(base, n_pol=npol, oversampling=beta, n_wplanes=1)
            wl = synth.make_workload(cfg)
            d = [torch.from_numpy(np.ascontiguousarray(x)).to(dev) for x in
                 (wl["uvw_m"], wl["baseline"], wl["vis"], wl["weights"])]
            n_bl = cfg.n_station * (cfg.n_station - 1) // 2
            for S in [int(x) for x in a.supports.split(",")]:
                if S > cfg.grid_n // 2:
                    continue
                sup = np.array([S], dtype=np.int32)
                per_step = n_bl * cfg.n_chan * S * S * npol
                n_t = int(max(1, min(cfg.n_time, a.max_updates // per_step)))
                rows = n_t * n_bl
                dd = [x[:rows] for x in d]
                g = Gridder(cfg.grid_n, wl["cell_rad"], 1, beta, S, npol, device=dev)
                g.allocate(sup, work_bytes=g.workspace_bytes(rows, cfg.n_chan))
                g.build_wkernels(0.0)
                if a.gather_min_support is not None:
                    g.set_gather_min_support(a.gather_min_support)
                g.grid_visibilities(dd[0], dd[1], wl["freqs_hz"], dd[2], dd[3])
                g.reset()
                for _ in range(a.steps):
                    g.grid_visibilities(dd[0], dd[1], wl["freqs_hz"], dd[2], dd[3])
                t = [g.timing(k) for k in range(a.steps)]
                sp = [g.gridder_split(k) for k in range(a.steps)]
                gridded, dropped, updates = g.stats()
                ms = float(np.mean([x[1] for x in t]))
                print(json.dumps({"workload": cfg.name, "support": S, "oversampling": beta, "n_pol": npol,
                                  "time_steps": n_t, "of_time_steps": cfg.n_time,
                                  "records_gridded": gridded // a.steps, "records_dropped": dropped // a.steps,
                                  "gridder_ms": ms, "ingest_ms": float(np.mean([x[0] for x in t])),
                                  "window_ms": float(np.mean([x[0] for x in sp])), "gather_ms": float(np.mean([x[1] for x in sp])),
                                  "updates_per_s": updates / a.steps / (ms * 1e-3),
                                  "records_per_s": gridded / a.steps / (ms * 1e-3)}), flush=True)
                g.close()
                del g


if __name__ == "__main__":
    main()
