"""ORACLE-side model of the gridder's atomic traffic - test/measurement infrastructure only.

Counts, from the oracle's own indices (oracle/ig_oracle.c orc_index), how many multi-polarised
PIXEL COMMITS a register-accumulating gridder needs when it walks every baseline's track in time
order, channel by channel ("commits per update"; Romein's scheme,
PAPER.md:730-742: a thread commits its sum when its grid point leaves the S x S window):

    window moves by (dx, dy), same support S :  S^2 - (S-|dx|)+ (S-|dy|)+   pixels leave -> commits
    support changes (or the record before was dropped) : the S_prev^2 held pixels all commit (:1349)
    end of a track : S_last^2

The count depends only on the inputs and on the paper's ordering, not on any CUDA kernel: bench.py
uses it for the roofline's atomic-byte term so that a kernel cannot raise its roofline fraction by
committing more often. This module imports only oracle/ and the seeded input generator.

    python -m oracle.track_commits            # rewrites oracle/track_commits.json (all five configs, both support laws)
"""
from __future__ import annotations

import json
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
if _ROOT not in sys.path:
    sys.path.insert(0, _ROOT)

from oracle import reference as orc  # noqa: E402
from paper_1403_4209_b200 import synth  # noqa: E402  (inputs only)

STORE = os.path.join(_HERE, "track_commits.json")
CLASSES = [(1, 15), (17, 31), (33, 63), (65, 127), (129, 511)]


def track_commits(X, Y, S, on, n_time, n_bl):
    """X, Y, S, on: [n_time*n_bl][nchan] (rows time-major, all baselines per time step).
    Returns (pixel commits, per-record commits array summed by support class, updates by class)."""
    nchan = X.shape[1]
    shp = (n_time, n_bl, nchan)
    X = X.reshape(shp); Y = Y.reshape(shp); S = S.reshape(shp).astype(np.int64); on = on.reshape(shp)
    S = np.where(on, S, 0)                     # a dropped record holds nothing
    total = 0
    by_class = np.zeros(len(CLASSES), dtype=np.int64)
    upd_class = np.zeros(len(CLASSES), dtype=np.int64)

    def add(sup, c):
        nonlocal total
        total += int(c.sum())
        for k, (lo, hi) in enumerate(CLASSES):
            m = (sup >= lo) & (sup <= hi)
            by_class[k] += int(c[m].sum())

    for t in range(n_time):
        s1 = S[t]
        for k, (lo, hi) in enumerate(CLASSES):
            upd_class[k] += int((s1[(s1 >= lo) & (s1 <= hi)] ** 2).sum())
        if t == 0:
            continue
        s0 = S[t - 1]
        dx = np.abs(X[t].astype(np.int64) - X[t - 1]); dy = np.abs(Y[t].astype(np.int64) - Y[t - 1])
        same = (s0 == s1)
        keep = np.clip(s0 - dx, 0, None) * np.clip(s0 - dy, 0, None)
        c = np.where(same, s0 * s0 - keep, s0 * s0)     # commits charged to the record that is left
        add(s0, c)
    sl = S[n_time - 1]
    add(sl, sl * sl)
    return total, by_class, upd_class


def model_config(index: int, law: str = "w"):
    cfg = synth.CONFIGS[index]
    wl = synth.make_workload(cfg, law, with_vis=False)
    sup = wl["supports"]
    idx = orc.index_records(wl["uvw_m"], wl["freqs_hz"], cfg.grid_n, wl["cell_rad"], cfg.oversampling,
                            cfg.n_wplanes, wl["w_max"], sup)
    n_bl = cfg.n_station * (cfg.n_station - 1) // 2
    on = (idx["flags"] & 2) != 0
    S = sup[idx["plane"]]
    commits, by_class, upd_class = track_commits(idx["X"], idx["Y"], S, on, cfg.n_time, n_bl)
    pix_updates = int((S.astype(np.int64)[on] ** 2).sum())
    return {"config": cfg.name, "support_law": law, "records": int(on.sum()), "pixel_updates": pix_updates,
            "pixel_commits": int(commits), "commits_per_update": commits / max(pix_updates, 1),
            "classes": [f"{lo}-{hi}" for lo, hi in CLASSES],
            "pixel_updates_by_support_class": [int(x) for x in upd_class],
            "pixel_commits_by_support_class": [int(x) for x in by_class]}


def load():
    with open(STORE) as f:
        return json.load(f)


def main():
    out = {"how": "python -m oracle.track_commits (oracle indices only; see module docstring)", "entries": []}
    which = [int(a) for a in sys.argv[1:]] or [0, 1, 2, 3, 4]
    for i in which:
        for law in ("w", "k"):
            e = model_config(i, law)
            print(json.dumps(e), flush=True)
            out["entries"].append(e)
    if len(which) == 5:
        with open(STORE, "w") as f:
            json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
