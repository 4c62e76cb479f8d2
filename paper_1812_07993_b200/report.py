"""Per-configuration throughput report (BASELINE.json configs[0..4]) -- `python -m paper_1812_07993_b200.report`.

For every configuration and force path: MD steps/s, pair-interactions/s (ordered within-cut-off evaluations,
algorithm-independent), executed pair tests/s, and for the all-pairs kernel the executed FP64/FP32 rate against the
FMA-chain peak measured in the same run.  Prints one markdown table; all inputs are the seeded synthetic
configurations of inputs.py.  (The CPU baseline for N <= 2^14 that configs[4] asks for is `bench.py --cpu-sweep`.)
"""
from __future__ import annotations

import argparse
import json
import sys


def time_steps(sim, n_steps, torch):
    sim.step(min(n_steps, 64))                       # warm-up (graph capture, first rebuilds)
    sim.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(sim.stream)
    sim.step(n_steps)
    b.record(sim.stream)
    sim.synchronize()
    return a.elapsed_time(b) * 1e-3 / n_steps


def measure(cfg, algo, precision, n_steps, torch, md, peaks):
    try:
        sim = md.Simulation(cfg, algo=algo, precision=precision)
    except md.MDError as e:
        if e.code == md.MD_ERR_UNSUPPORTED:
            return None
        raise
    sec = time_steps(sim, n_steps, torch)
    e = sim.energy()
    tests = sim.pair_tests()
    inter = 2 * e["pairs_vv"] + e["pairs_vw"]
    nv, nw = cfg["n_vapor"], cfg["n_wall"]
    # compulsory state traffic of a fully fused step: read r, v and write r', v' = 4 * dim reals per particle
    state_bytes = 4 * cfg["dim"] * (precision // 8) * nv
    row = dict(config=cfg["name"], n_vapor=nv, n_wall=nw, algo=sim.info()["algo"], precision=precision,
               steps_timed=n_steps, md_steps_per_s=1.0 / sec, pair_interactions_per_s=inter / sec,
               pair_tests_per_s=tests / sec, allpairs_equivalent_per_s=nv * (nv - 1.0 + nw) / sec, us_per_step=sec * 1e6,
               state_gbs=state_bytes / sec * 1e-9, state_frac_of_copy_peak=state_bytes / sec * 1e-9 / peaks["copy_gbs"])
    if algo == "allpairs":
        flops = 6.0                                   # executed per test (3 fma): DESIGN.md section 5
        peak = peaks["fp64_tflops"] if precision == 64 else peaks["fp32_tflops"]
        row["alu_tflops"] = tests * flops / sec * 1e-12
        row["alu_frac_of_measured_peak"] = row["alu_tflops"] / peak
    sim.close()
    return row


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="0,1,2,3,4,5", help="0-4: BASELINE.json configs; 5: the paper's problem sizes; "
                    "6: the paper's N sweeps of Tables 2-3 (N_pore = 100 ... 1500)")
    ap.add_argument("--max-log2n", type=int, default=20)
    ap.add_argument("--min-log2n", type=int, default=10)
    ap.add_argument("--paths", default="allpairs,cells,verlet", help="force paths to run (subset)")
    ap.add_argument("--precisions", default="64,32", help="config 4 precisions to run (subset)")
    ap.add_argument("--steps", type=int, default=0, help="override the number of timed steps of every row (0: per-config defaults)")
    ap.add_argument("--json", default="")
    ap.add_argument("--split", default="", help="instead of the table: the persistent kernel's own timers (md_profile_step) for "
                    "these workloads, comma separated: cfg0, cfg1, cfg2, cfg3, 2pK (config 4 at 2^K); --steps per launch "
                    "(default 2000) after --split-warmup steps (default 500)")
    ap.add_argument("--split-warmup", type=int, default=500)
    args = ap.parse_args()
    import torch

    from . import inputs as I
    from . import md

    if not torch.cuda.is_available():
        raise SystemExit("report: no CUDA device; the CUDA path has no fallback")
    if args.split:
        print("| workload | us per step: total = phase + barrier wait + list events | full rebuilds (us each: bin / scan / scatter / build) "
              "| prunes (us each) |\n|---|---|---|---|")
        for name in args.split.split(","):
            cfg = {"cfg0": I.config0, "cfg1": I.config1, "cfg2": I.config2, "cfg3": lambda: I.config3("cone")}.get(
                name, lambda: I.config4(int(name[2:])))()
            sim = md.Simulation(cfg, algo="verlet")
            done = 0
            while done < args.split_warmup:                      # long warm-ups (the film on the pore wall) in 20,000-step launches
                n = min(20000, args.split_warmup - done)
                sim.step(n)
                done += n
            n = args.steps or 2000
            k = sim.profile_step(n)
            us = [x * 1e3 / n for x in k["ms"]]
            print("| %s after %d steps | %.2f = %.2f + %.2f + %.2f | %d (%s) | %d (%.1f) |" % (
                name, args.split_warmup, k["total_ms"] * 1e3 / n, us[0], us[1], us[2], k["rebuilds"],
                " / ".join("%.1f" % (x * 1e3 / max(k["rebuilds"], 1)) for x in k["rebuild_ms"]), k["prunes"],
                k["prune_ms"] * 1e3 / max(k["prunes"], 1)), flush=True)
            sim.close()
        return
    peaks = md.measure_peaks()
    want = {int(x) for x in args.configs.split(",")}
    rows = []

    paths = set(args.paths.split(","))
    precisions = {int(x) for x in args.precisions.split(",")}

    def add(cfg, algo, precision, n_steps):
        if algo not in paths or precision not in precisions:
            return
        r = measure(cfg, algo, precision, args.steps or n_steps, torch, md, peaks)
        if r:
            rows.append(r)
            print("  %-22s %-8s fp%d  %10.0f steps/s" % (r["config"], r["algo"], precision, r["md_steps_per_s"]), file=sys.stderr)

    if 0 in want:
        cfg = I.config0()
        for algo in ("allpairs", "cells", "verlet"):
            add(cfg, algo, 64, 2000)
    if 1 in want:
        cfg = I.config1()
        for algo in ("cells", "verlet"):
            add(cfg, algo, 64, 4000)
    if 2 in want:
        cfg = I.config2()
        for algo in ("cells", "verlet"):
            add(cfg, algo, 64, 4000)
        add(cfg, "allpairs", 64, 20)
    if 3 in want:
        for shape in ("cone", "inkbottle", "slit"):
            cfg = I.config3(shape)
            for algo in ("cells", "verlet"):
                add(cfg, algo, 64, 2000)
    if 5 in want:      # the paper's own problem sizes, context for its Tables 1 and 4
        for dim in (2, 3):
            cfg = I.paper_size(dim)
            for algo in ("allpairs", "cells", "verlet"):
                add(cfg, algo, 64, 2000)
            add(I.paper_geometry(dim), "allpairs", 64, 2000)      # the paper's geometry, units and 2000 steps (NEXT-3)
    if 6 in want:      # Tables 2-3: N molecules in the pore, N_tot = 5.2 N (2D) / 2.8 N (3D), 2000 steps
        for dim in (2, 3):
            for n_pore in range(100, 1501, 100):
                add(I.paper_geometry(dim, n_pore=n_pore), "allpairs", 64, 2000)
    if 4 in want:
        for log2n in range(args.min_log2n, args.max_log2n + 1, 2):
            cfg = I.config4(log2n)
            for precision in (64, 32):
                for algo in ("cells", "verlet"):
                    add(cfg, algo, precision, 1000)
                # all-pairs cost grows as N^2: 1000 steps up to 2^14, fewer beyond (stated in the table)
                ap_steps = {10: 1000, 12: 1000, 14: 1000, 16: 100, 18: 10, 20: 2}[log2n]
                add(cfg, "allpairs", precision, ap_steps)
    print("peaks measured in this run: FP64 %.1f TFLOP/s, FP32 %.1f TFLOP/s, copy %.0f GB/s\n" %
          (peaks["fp64_tflops"], peaks["fp32_tflops"], peaks["copy_gbs"]))
    print("Rates (SURVEY 8(d)): pair-interactions/s = ordered within-cut-off evaluations; pair tests/s = ordered distance tests "
          "executed; all-pairs-equivalent/s = N_v (N_v - 1 + N_w) x steps/s (comparable with the paper's derived 1-2.8e9); "
          "state GB/s = compulsory bytes of a fully fused step (read r, v; write r', v': 96 B per particle in 3D fp64) x steps/s, "
          "against the device-copy GB/s measured in this run.\n")
    print("| config | N_v | N_w | path | fp | steps timed | MD steps/s | us/step | pair-interactions/s | pair tests/s | all-pairs-equivalent/s | "
          "state GB/s (frac of copy peak) | ALU TFLOP/s (frac of measured peak) |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for r in rows:
        alu = "%.2f (%.3f)" % (r["alu_tflops"], r["alu_frac_of_measured_peak"]) if "alu_tflops" in r else ""
        print("| %s | %d | %d | %s | %d | %d | %.4g | %.4g | %.4g | %.4g | %.4g | %.1f (%.3f) | %s |" %
              (r["config"], r["n_vapor"], r["n_wall"], r["algo"], r["precision"], r["steps_timed"], r["md_steps_per_s"],
               r["us_per_step"], r["pair_interactions_per_s"], r["pair_tests_per_s"], r["allpairs_equivalent_per_s"],
               r["state_gbs"], r["state_frac_of_copy_peak"], alu))
    if args.json:
        with open(args.json, "w") as fh:
            json.dump(dict(peaks=peaks, rows=rows), fh)


if __name__ == "__main__":
    main()
