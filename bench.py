#!/usr/bin/env python
"""bench.py - one JSON line for the gridding hot path on N B200s (contract in the task statement).

A "step" is one pass of the whole hot path (ingest A1-A3 + gridder C = one ig_grid call) over the
full synthetic workload of the chosen BASELINE.json configuration. `value` = grid-point updates/s
(sum S^2 * n_pol over gridded records / device time, sec 5.3.1) with inputs resident in
HBM; `e2e` = the same through ig_grid_host with pinned host buffers, copies inside the timed region.
`--impl reference` times the fp64 CPU oracle (oracle/), as it stands, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1403_4209_b200 import synth  # noqa: E402  (data only)

METRIC = "grid_point_updates_per_s"
UNIT = "updates/s"
WORKLOADS = ["cfg1_tiny_plain", "cfg2_small_wproj", "cfg3_medium", "cfg4_large", "cfg5_stress"]


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=int(os.environ.get("IG_BENCH_CONFIG", "5")),
                    help="BASELINE.json configuration 1..5 (default 5, the largest W-projection config the target is quoted on)")
    ap.add_argument("--support-law", default="w", choices=["w", "k"])
    ap.add_argument("--no-compress", action="store_true", help="switch compression off (thesis: real vs total rate)")
    ap.add_argument("--host-slices", type=int, default=8, help="ig_grid_host: slices copied while the previous one is gridded")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=20.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(config):
    """DRAM bytes per launch of k_gridder from the committed ncu capture of this configuration
    (profiles/traffic.csv: config,kernel,dram_read_bytes,dram_write_bytes,capture), or None."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(path) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) >= 4 and c[0] == str(config) and c[1] == "k_gridder":
                    return float(c[2]) + float(c[3])
    except OSError:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_oracle_sample(cfg, law, target_s):
    """Time the oracle (index + gridding, fp64, OpenMP row bands) on the first whole time steps of the
    workload. The kernel-bank VALUES are seeded random numbers of the right shape: the oracle's own numpy
    bank builder would take minutes for hundreds of planes, and the record loop's work does not depend on
    them. Returns dict(value, cores, sample, seconds, updates, records)."""
    from oracle import reference as orc
    orc.build()
    n_bl = cfg.n_station * (cfg.n_station - 1) // 2
    wl_full = synth.make_workload(cfg, law, with_vis=False)
    sup = wl_full["supports"]
    mean_s2 = float((sup.astype(np.float64) ** 2).mean())
    # aim at target_s assuming ~2e8 fp64 complex updates/s/core as a first guess
    cores = orc.threads()
    guess_updates = 2e8 * cores * target_s
    per_step = n_bl * cfg.n_chan * mean_s2 * cfg.n_pol * 0.35
    n_t = int(max(1, min(cfg.n_time, guess_updates // max(per_step, 1))))
    rows = n_t * n_bl
    uvw, bl = wl_full["uvw_m"][:rows], wl_full["baseline"][:rows]
    rng = np.random.Generator(np.random.Philox(99))
    shape = (rows, cfg.n_chan, cfg.n_pol)
    vis = (rng.standard_normal(shape + (2,), dtype=np.float32)).view(np.complex64)[..., 0]
    wt = (0.5 + 0.5 * rng.random(shape, dtype=np.float32)).astype(np.float32)
    b2 = cfg.oversampling ** 2
    off = np.zeros(sup.size, dtype=np.int64)
    off[1:] = np.cumsum(sup[:-1].astype(np.int64) ** 2 * b2)
    n_el = int((sup.astype(np.int64) ** 2).sum() * b2)
    bank = np.empty(n_el, dtype=np.complex128)
    bank.view(np.float64)[:] = rng.random(2 * n_el)
    grid = np.zeros((cfg.grid_n, cfg.grid_n, cfg.n_pol), dtype=np.complex128)
    t0 = time.perf_counter()
    idx = orc.index_records(uvw, wl_full["freqs_hz"], cfg.grid_n, wl_full["cell_rad"], cfg.oversampling,
                            cfg.n_wplanes, wl_full["w_max"], sup)
    _, _, stats = orc.grid_records(idx, vis, wt, cfg.grid_n, cfg.oversampling, sup, bank, off, grid=grid)
    dt = time.perf_counter() - t0
    return dict(value=float(stats[2]) / dt, cores=cores, seconds=dt, updates=int(stats[2]), records=int(stats[0]),
                sample=f"oracle orc_index+orc_grid (fp64, {cores} OpenMP threads) on the first {n_t} of {cfg.n_time} time "
                       f"steps x all {n_bl} baselines x {cfg.n_chan} channels = {int(stats[0])} records of {cfg.name}; "
                       f"kernel-bank values seeded random (timing only)")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = synth.CONFIGS[args.config - 1]
    times, last = [], None
    for i in range(args.warmup + args.steps):
        last = cpu_oracle_sample(cfg, args.support_law, min(args.cpu_seconds, 8.0))
        if i >= args.warmup:
            times.append(last)
    upd = sum(t["updates"] for t in times)
    sec = sum(t["seconds"] for t in times)
    val = upd / sec
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sec / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config - 1], "support_law": args.support_law, "sample": last["sample"]},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import torch
    from paper_1403_4209_b200 import build as igbuild
    from paper_1403_4209_b200.binding import Gridder

    from paper_1403_4209_b200.dist import Ranks
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    ranks = Ranks(backend="nccl", device=dev)
    world, rank = ranks.world, ranks.rank
    if rank == 0:
        igbuild.build()
    ranks.barrier()

    def barrier():
        ranks.barrier()
        torch.cuda.synchronize(dev)

    max_over_ranks = ranks.max_over_ranks

    cfg = synth.CONFIGS[args.config - 1]
    t_gen = time.perf_counter()
    wl = synth.make_workload(cfg, args.support_law)       # replicas only: every rank grids the same workload
    t_gen = time.perf_counter() - t_gen
    sup = wl["supports"]
    nrow, nchan, npol = wl["uvw_m"].shape[0], cfg.n_chan, cfg.n_pol
    g = Gridder(cfg.grid_n, wl["cell_rad"], cfg.n_wplanes, cfg.oversampling, int(sup.max()), npol, device=str(dev))
    g.allocate(sup, work_bytes=g.workspace_bytes(nrow, nchan, host=not args.no_e2e))
    t0 = time.perf_counter()
    g.build_wkernels(wl["w_max"])
    torch.cuda.synchronize(dev)
    t_bank = time.perf_counter() - t0
    fp32_peak = g.measure_fp32_peak()
    g.set_compression(not args.no_compress)
    g.set_host_slices(args.host_slices)

    pin = (lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()) if not args.no_e2e else None
    vis_f = np.ascontiguousarray(wl["vis"]).view(np.float32).reshape(nrow, nchan, npol, 2)
    host = dict(uvw=wl["uvw_m"], bl=wl["baseline"], vis=vis_f, wt=wl["weights"])
    if pin:
        host = {k: pin(v) for k, v in host.items()}
        d = {k: v.to(dev, non_blocking=True) for k, v in host.items()}
    else:
        d = {k: torch.from_numpy(v).to(dev) for k, v in host.items()}
    freqs = wl["freqs_hz"]
    h2d_bytes = sum(int(v.numel() * v.element_size()) if hasattr(v, "numel") else v.nbytes for v in host.values()) + freqs.nbytes

    def step():
        g.grid_visibilities(d["uvw"], d["bl"], freqs, d["vis"], d["wt"])

    # one counted pass from a zero grid: statistics of ONE step (also the first warm-up)
    g.reset()
    g.set_commit_counting(True)
    step()
    gridded, dropped, updates = g.stats()
    commits = g.commits()
    compressed = g.compressed()
    g.set_commit_counting(False)
    touched = g.touched_pixels()
    launches_per_step = g.last_launches()
    for _ in range(max(0, args.warmup - 1)):
        step()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    clocks = sampler.stop() if rank == 0 else None
    split = [g.timing(k) for k in range(min(args.steps, 64))]
    ingest_ms = float(np.mean([s[0] for s in split]))
    gridder_ms = float(np.mean([s[1] for s in split]))
    ms_step = ms_total / args.steps
    value = world * updates / (ms_step * 1e-3)

    # end to end: host buffers through ig_grid_host, H2D copies and the D2H read of the step's result inside
    e2e = None
    if not args.no_e2e:
        def e2e_step():
            g.grid_visibilities_host(host["uvw"], host["bl"], freqs, host["vis"], host["wt"])
            return g.stats()                    # D2H read of the step's result (eq 4.17 counters), synchronises
        e2e_step()
        n_e2e = max(1, min(args.steps, 3))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        torch.cuda.synchronize(dev)
        dt = max_over_ranks(time.perf_counter() - t0) / n_e2e
        e2e = {"value": world * updates / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d_bytes), "d2h_bytes_per_step": 56,
               "ms_per_step": dt * 1e3, "steps": n_e2e, "host_slices": args.host_slices,
               "how": "ig_grid_host from pinned host buffers, slice k+1 copied while slice k is gridded, then ig_get_stats"}

    if rank != 0:
        ranks.close()
        return

    # ---- roofline of the dominant kernel (k_gridder), DESIGN.md "Roofline" -------------------------
    hbm_peak, peak_src = peaks()
    stride = 48 if npol == 4 else 32
    n_chunks = ((nrow + 127) // 128) * nchan
    bank_bytes = int((sup.astype(np.int64) ** 2).sum()) * cfg.oversampling ** 2 * 8
    alg_bytes = n_chunks * 128 * stride + bank_bytes + commits * 8 * npol + touched * 8 * npol * 2
    t_byte = alg_bytes / (hbm_peak * 1e9)
    flops = 8.0 * updates
    t_flop = flops / (fp32_peak * 1e12)
    gs = gridder_ms * 1e-3
    if t_byte >= t_flop:
        roof = {"bound": "hbm", "achieved": alg_bytes / gs / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": t_byte / gs, "traffic": ncu_traffic(args.config), "peak_source": peak_src}
    else:
        roof = {"bound": "alu", "achieved": flops / gs / 1e12, "peak": fp32_peak, "unit": "TFLOP/s",
                "frac": t_flop / gs, "traffic": ncu_traffic(args.config), "peak_source": "measured live: ig_measure_fp32_peak (FFMA loop)"}
    roof.update({"kernel": "k_gridder", "kernel_ms": gridder_ms, "t_flop_ms": t_flop * 1e3, "t_byte_ms": t_byte * 1e3,
                 "algorithmic_bytes": int(alg_bytes), "flops": flops, "fp32_peak_tflops": fp32_peak, "hbm_peak_gbs": hbm_peak,
                 "commits": commits, "touched_pixels": touched})

    cpu = None
    if not args.no_cpu and world == 1:
        c = cpu_oracle_sample(cfg, args.support_law, args.cpu_seconds)
        cpu = {"value": c["value"], "unit": UNIT, "cores": c["cores"], "kind": "oracle", "sample": c["sample"],
               "seconds": c["seconds"]}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config - 1], "grid_n": cfg.grid_n, "n_pol": npol, "n_chan": nchan, "rows": int(nrow),
                   "records": int(nrow) * nchan, "w_planes": cfg.n_wplanes, "support": [int(sup.min()), int(sup.max())],
                   "support_law": args.support_law, "oversampling": cfg.oversampling, "parallelism": f"replicas x{world}",
                   "l2": "inputs (%.1f GB) larger than L2; no flush needed" % (h2d_bytes / 1e9)},
        "visibilities_per_s": world * gridded / (ms_step * 1e-3),
        "records_gridded": gridded, "records_dropped": dropped, "updates_per_step": updates,
        "compression": {"enabled": not args.no_compress, "records_compressed": compressed,
                        "note": "value counts every gridded record (thesis total rate, PAPER.md:1767); "
                                "real rate = value * (1 - records_compressed / records_gridded)"},
        "ingest_ms": ingest_ms, "gridder_ms": gridder_ms, "gridder_updates_per_s": updates / gs,
        "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
        "clocks": clocks, "setup": {"generate_s": t_gen, "build_wkernels_s": t_bank},
        "context": "thesis GTX 680: ~50 G updates/s real rate, Romein 93 G (PAPER.md:742,:1986) - other hardware, not a target",
    }
    print(json.dumps(out))
    ranks.close()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
