#!/usr/bin/env python
"""bench.py -- pair-interactions/s and MD steps/s on the 3D 65,536-particle cylindrical pore (BASELINE.json
configs[2]), one replica per GPU (replicas only, no data-path collective).

One bench "step" = `--inner` velocity-Verlet timesteps (rows a1-a4 of DESIGN.md every timestep) followed by one
md_energy call (row a5).  `value` times that with the state resident in HBM; `e2e` times
md_create(host arrays) -> md_step -> md_get_state(host arrays) + md_energy through the C ABI.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--inner M] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "pair-interactions/s"
WORKLOAD = "cfg2_cyl3d_64k: 3D cylindrical pore, 65536 vapor + 1240 wall particles, 110^3 box, fp64, cell list"


def peaks_file():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh), "measured"
    except OSError:
        return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) >= 7 and r[3 + k] == "Active" for r in self.rows)]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def oracle_sample(cfg, n_steps):
    """Times the CPU oracle (cell-list variant, as it stands) for n_steps timesteps of cfg."""
    from oracle import md_oracle as O

    O.forces(cfg, cells=True)                                   # build / page in
    t0 = time.perf_counter()
    out = O.run(cfg, n_steps, cells=True, history=True)
    dt = time.perf_counter() - t0
    h = out["hist"]
    inter = float((h[1:, 3] + h[1:, 4]).sum())                  # ordered vv hits + vw hits per evaluated step
    return dt, inter, O.n_threads()


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    from paper_1812_07993_b200 import inputs as I

    cfg = I.config2()
    per = max(1, args.ref_inner)
    for _ in range(args.warmup):
        oracle_sample(cfg, 1)
    tot_t, tot_i = 0.0, 0.0
    cores = 1
    for _ in range(args.steps):
        dt, inter, cores = oracle_sample(cfg, per)
        tot_t += dt
        tot_i += inter
    val = tot_i / tot_t
    sample = "%d bench steps x %d oracle (CPU cell-list) timesteps of cfg2 from t=0" % (args.steps, per)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": METRIC, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "md_steps_per_s": args.steps * per / tot_t, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "md_steps_per_bench_step": per},
            "cpu_baseline": {"value": val, "unit": METRIC, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
