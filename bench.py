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
WORKLOAD = ("cfg2_cyl3d_64k: 3D cylindrical pore, 65536 vapor + 1240 wall particles, 110^3 box, fp64, "
            "cell list cached as a Verlet list (MD_FORCE_AUTO)")
STATE_BYTES = 96       # compulsory bytes per particle-step of a fully fused step, 3D fp64 (read r, v; write r', v')
ALGO = "auto"      # resolves to the persistent Verlet-list kernel on this workload (md.h: MD_FORCE_AUTO)


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
    from paper_1812_07993_b200 import replicas

    return replicas.dist_env()


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


def run_ours(args):
    import torch

    from paper_1812_07993_b200 import inputs as I
    from paper_1812_07993_b200 import md

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no fallback")
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    md.load_library()
    from paper_1812_07993_b200 import replicas

    cfg = replicas.replica_config(rank)                         # one independent replica per rank
    nv, nw, dim = cfg["n_vapor"], cfg["n_wall"], cfg["dim"]
    inner = args.inner

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def max_over_ranks(x):
        return replicas.max_over_ranks(x, dev)

    def sum_over_ranks(x):
        return replicas.sum_over_ranks(x, dev)

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    # ---------------- device-resident arm -------------------------------------------------
    sim = md.Simulation(cfg, algo=ALGO, device=dev)
    info = sim.info()
    for _ in range(args.warmup):
        sim.step(inner)
        sim.energy()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev = [tuple(torch.cuda.Event(enable_timing=True) for _ in range(3)) for _ in range(args.steps)]
    inter = 0.0
    e = sim.energy()
    hits_before = 2 * e["pairs_vv"] + e["pairs_vw"]
    barrier()
    for a, m, b in ev:
        flush.zero_()                                               # L2 flush between timed iterations (untimed)
        sim.stream.wait_stream(torch.cuda.current_stream(dev))
        a.record(sim.stream)
        sim.step(inner)                                             # a1-a4: ONE launch of k_md_run (persistent path)
        m.record(sim.stream)
        e = sim.energy()                                            # a5; synchronises the stream
        b.record(sim.stream)
        hits = 2 * e["pairs_vv"] + e["pairs_vw"]                    # ordered within-cut-off evaluations per time step,
        inter += 0.5 * (hits_before + hits) * inner                 # mean of the counts at both ends of the chunk
        hits_before = hits
    barrier()
    t_dev = max_over_ranks(sum(a.elapsed_time(b) for a, m, b in ev) * 1e-3)
    t_run = sum(a.elapsed_time(m) for a, m, b in ev) * 1e-3        # the k_md_run launches alone (this rank)
    clocks = sampler.stop() if rank == 0 else None
    inter_all = sum_over_ranks(inter)
    value = inter_all / t_dev
    steps_per_s = args.steps * inner / t_dev                        # per replica (all replicas advance together)
    persistent = info["algo"] == "verlet"
    launches = args.steps * ((1 if persistent else inner * info["kernels_per_step"]) + 3)   # + the three energy kernels

    # ---------------- end-to-end arm: host arrays in, host arrays out, through the C ABI ----
    host = {k: torch.from_numpy(np.ascontiguousarray(cfg[k])).pin_memory().numpy() for k in ("pos", "vel", "wall")}
    ecfg = dict(cfg)
    ecfg.update(host)
    stream = torch.cuda.Stream(device=dev)
    e2e_inter = 0.0
    s0 = md.Simulation(ecfg, algo=ALGO, device=dev, stream=stream)
    e = s0.energy()
    hits0 = 2 * e["pairs_vv"] + e["pairs_vw"]                       # every end-to-end step starts from the same t = 0 state
    s0.close()

    def e2e_step():
        s2 = md.Simulation(ecfg, algo=ALGO, device=dev, stream=stream)    # H2D of pos, vel, wall
        s2.step(inner)
        st = s2.get_state(force=False, pe=False)                              # D2H of pos, vel
        e = s2.energy()
        s2.close()
        return 0.5 * (hits0 + 2 * e["pairs_vv"] + e["pairs_vw"]) * inner, st

    for _ in range(args.warmup):        # untimed, like the device arm's warm-up: on a fresh box the first end-to-end steps
        e2e_step()                      # pay for page-locking and first-use set-up (measured 24-31 ms against 19.4)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_inter += e2e_step()[0]
    barrier()
    t_e2e = max_over_ranks(time.perf_counter() - t0)
    e2e_value = sum_over_ranks(e2e_inter) / t_e2e
    h2d = 8 * dim * (2 * nv + nw)
    d2h = 8 * dim * 2 * nv + 6 * 8 + 4

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---------------- roofline of the dominant kernel, measured live (rank 0) --------------
    pk, pk_src = peaks_file()
    tests = sim.pair_tests()
    ncell = int(np.prod(info["n_cells"]))
    if persistent:
        # k_md_run is the whole timed step but for the three energy kernels: its launches were timed above with CUDA
        # events on the stream they run on.  achieved = algorithmic bytes / that time, with SURVEY 8(d)'s compulsory
        # 96 B per particle-step; the bytes this LAYOUT moves per particle-step (32-byte positions with the path length
        # in w, read and written; velocities read and written; the list: count word + 4 B per entry) are given beside it
        top_name = "k_md_run (persistent: %d time steps per launch)" % inner
        t_top = t_run / args.steps
        alg = STATE_BYTES * nv * inner
        layout = (nv * (64 + 48 + 4) + 4 * tests) * inner
        shares = {"k_md_run": t_run / (sum(a.elapsed_time(b) for a, m, b in ev) * 1e-3)}
        traffic = None
        kt = sim.profile_step(inner)                                # in-kernel split of one more launch (after the timed region)
        extra = {"time_steps_per_launch": inner, "us_per_time_step": t_top * 1e6 / inner, "layout_bytes_per_launch": layout,
                 "traffic_source": "profiles/r02_k_md_run.md (ncu --set full of one launch: dram__bytes_read.sum + dram__bytes_write.sum)",
                 "in_kernel_split_of_one_more_launch_us_per_time_step": {
                     "step_phases": kt["ms"][0] * 1e3 / inner, "grid_barriers": kt["ms"][1] * 1e3 / inner,
                     "rebuilds": kt["ms"][2] * 1e3 / inner, "rebuilds_in_launch": kt["rebuilds"],
                     "rebuild_us_each_bin_scan_scatter_build": [x * 1e3 / max(kt["rebuilds"], 1) for x in kt["rebuild_ms"]]}}
    else:
        prof_steps = 200
        sim.profile_step(20)
        kt = sim.profile_step(prof_steps)
        names = ["kick_drift_bin", "scan", "scatter", "force_kick"]
        shares = {n: kt["ms"][k] / max(kt["total_ms"], 1e-12) for k, n in enumerate(names)}
        top = max(range(4), key=lambda k: kt["ms"][k])
        alg_bytes = {0: 144 * nv, 1: 12 * ncell, 2: 128 * nv + 4 * ncell, 3: 104 * nv + 4 * (ncell + 1)}
        top_name, t_top, alg = names[top], kt["ms"][top] * 1e-3 / kt["launches"][top], alg_bytes[top]
        extra, traffic = {}, None
    achieved = alg / t_top * 1e-9
    roofline = {"kernel": top_name, "bound": "hbm", "achieved": achieved, "peak": pk["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / pk["hbm_gbs"], "traffic": traffic, "peak_source": pk_src + " (MEASURED_PEAKS.json hbm_gbs)",
                "algorithmic_bytes_per_launch": alg, "us_per_launch": t_top * 1e6, "kernel_share_of_step": shares,
                "note": "the 4.7 MB state is L2-resident across time steps, so the step is bound by L2 latency and the "
                        "grid barrier, not by HBM: a low fraction here is expected (DESIGN.md)"}
    roofline.update(extra)
    sim.close()

    # the counting-sort cell path rebuilt every step (MD_FORCE_CELLS), same workload, for comparison
    sim_c = md.Simulation(cfg, algo="cells", device=dev)
    sim_c.step(64)
    sim_c.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(sim_c.stream)
    sim_c.step(512)
    e1.record(sim_c.stream)
    sim_c.synchronize()
    cells_path = {"md_steps_per_s": 512 / (e0.elapsed_time(e1) * 1e-3), "pair_tests_per_timestep": sim_c.pair_tests(),
                  "kernels_per_step": sim_c.info()["kernels_per_step"]}
    sim_c.close()

    # FP64 roofline of the all-pairs force kernel at the same N (north_star: % of FP64 peak, measured in the same run)
    peaks = md.measure_peaks(device=dev)
    sim_ap = md.Simulation(cfg, algo="allpairs", device=dev)
    sim_ap.profile_step(1)
    ap = sim_ap.profile_step(args.allpairs_steps)
    t_ap = ap["ms"][3] * 1e-3 / ap["launches"][3]
    ap_tests = sim_ap.pair_tests()
    sim_ap.close()
    flops_per_test = 6.0            # executed per test: 3 DFMA (md_allpairs.cuh)
    ap_tflops = ap_tests * flops_per_test / t_ap * 1e-12
    allpairs = {"kernel": "force_allpairs", "bound": "alu", "pair_tests_per_s": ap_tests / t_ap,
                "achieved": ap_tflops, "peak": peaks["fp64_tflops"], "unit": "TFLOP/s",
                "frac": ap_tflops / peaks["fp64_tflops"], "flops_per_test": flops_per_test,
                "ms_per_launch": t_ap * 1e3, "peak_source": "DFMA chain measured in this run (md_measure_peaks)",
                "md_steps_per_s": 1.0 / (ap["total_ms"] * 1e-3 / ap["steps"]),
                "note": "tests include this step's periodic ghost entries; slot 3 = force kernel + the 3 us kick kernel"}

    # ---------------- CPU baseline: the oracle as it stands, bounded sample -----------------
    dt_cpu, inter_cpu, cores = oracle_sample(I.config2(), args.cpu_steps)
    cpu = {"value": inter_cpu / dt_cpu, "unit": METRIC, "cores": cores, "kind": "oracle",
           "md_steps_per_s": args.cpu_steps / dt_cpu,
           "sample": "%d timesteps of cfg2 from t=0 with the oracle's CPU cell-list variant" % args.cpu_steps}

    line = {"metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_dev / args.steps, "md_steps_per_s": steps_per_s,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "md_steps_per_bench_step": inner, "replicas": world,
                       "force_algo": info["algo"], "n_cells": info["n_cells"],
                       "l2": "256 MiB buffer written between timed iterations (L2 flush); inside an iteration the "
                             "4.7 MB state stays L2-resident across timesteps, as in any MD time loop",
                       "pair_tests_per_timestep": tests},
            "pair_tests_per_s": tests * steps_per_s * world,
            "allpairs_equivalent_per_s": float(nv) * (nv - 1.0 + nw) * steps_per_s * world, "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": METRIC, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": 1e3 * t_e2e / args.steps},
            "gpu_launches": launches, "roofline": roofline, "cells_every_step_path": cells_path,
            "roofline_allpairs_fp64": allpairs,
            "measured_peaks_this_run": peaks, "cpu_baseline": cpu}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_cpu_sweep():
    """CPU baseline of BASELINE.json configs[4]: the brute-force oracle on the host cores for N_v <= 2^14."""
    from oracle import md_oracle as O
    from paper_1812_07993_b200 import inputs as I

    print("| N_v | N_w | cores | s per step | ordered pair tests/s |\n|---|---|---|---|---|")
    for log2n in (10, 12, 14):
        cfg = I.config4(log2n)
        O.forces(cfg)
        n = 3
        t0 = time.perf_counter()
        O.run(cfg, n)
        sec = (time.perf_counter() - t0) / (n + 1)              # n steps + the initial force evaluation
        nv, nw = cfg["n_vapor"], cfg["n_wall"]
        print("| %d | %d | %d | %.4g | %.4g |" % (nv, nw, O.n_threads(), sec, nv * (nv - 1 + nw) / sec))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--inner", type=int, default=2000, help="MD timesteps per bench step")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-inner", type=int, default=20, help="oracle timesteps per bench step (--impl reference)")
    ap.add_argument("--cpu-steps", type=int, default=3000, help="oracle timesteps of the cpu_baseline sample (~15 s on 16 cores)")
    ap.add_argument("--allpairs-steps", type=int, default=10)
    ap.add_argument("--cpu-sweep", action="store_true", help="time the brute-force oracle for N_v = 2^10, 2^12, 2^14")
    args = ap.parse_args()
    if args.gpus > 1 and "RANK" not in os.environ and not args.cpu_sweep and args.impl == "ours":
        # started plainly: become the N-rank job the contract describes (one process per GPU, NCCL for the barrier)
        import socket

        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execvp(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
                                   "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    if args.cpu_sweep:
        run_cpu_sweep()
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
