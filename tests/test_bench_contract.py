"""The bench line committed under profiles/ carries every key of the bench contract (CPU-side check of the JSON
shape; the numbers themselves come from the GPU box)."""
import json
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _line(name):
    with open(os.path.join(ROOT, "profiles", name)) as fh:
        return json.loads(fh.read().strip().splitlines()[-1])


def test_our_arm_has_every_contract_key():
    d = _line("bench_r02_final.json.txt")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["metric"] == "pair-interactions/s" and d["higher_is_better"] is True and d["scaling"] == "weak"
    assert d["vs_baseline"] is None and d["dtype"] == "f64" and d["data"] == "synthetic" and d["warmup"] >= 3
    assert "workload" in d["config"] and "model" not in d["config"]
    assert {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"} <= set(d["e2e"])
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0 and d["e2e"]["value"] != d["value"]
    r = d["roofline"]
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(r) and r["bound"] in ("hbm", "tensor", "alu")
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    # the dominant kernel is timed inside the timed region: it cannot take longer than the step that contains it, and
    # its achieved GB/s is SURVEY 8(d)'s 96 B per particle-step over that time
    assert r["us_per_launch"] <= d["ms_per_step"] * 1e3
    nv, inner = 65536, d["config"]["md_steps_per_bench_step"]
    assert r["algorithmic_bytes_per_launch"] == 96 * nv * inner
    assert abs(r["achieved"] - 96 * nv * inner / (r["us_per_launch"] * 1e-6) * 1e-9) < 1e-6 * r["achieved"]
    assert r["traffic"] is None or r["traffic"] > 0
    assert "allpairs_equivalent_per_s" in d
    c = d["cpu_baseline"]
    assert {"value", "unit", "cores", "kind", "sample"} <= set(c) and c["kind"] == "oracle"
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"]) and d["gpu_launches"] > 0
    assert not set(d["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}


def test_reference_arm_line():
    d = _line("bench_r02_final_reference_arm.json.txt")
    assert d["impl"] == "reference" and d["metric"] == "pair-interactions/s" and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]


def test_plain_start_with_gpus_n_spawns_n_ranks(monkeypatch):
    """`python bench.py --gpus 8` started without torchrun must become the 8-rank job itself (one process per GPU)."""
    import importlib.util
    import sys

    spec = importlib.util.spec_from_file_location("bench_under_test", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    seen = {}

    def fake_exec(prog, argv):
        seen["argv"] = argv
        raise SystemExit(0)

    monkeypatch.setattr(bench.os, "execvp", fake_exec)
    monkeypatch.delenv("RANK", raising=False)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "8", "--steps", "2", "--warmup", "3"])
    try:
        bench.main()
    except SystemExit:
        pass
    argv = seen["argv"]
    assert "torch.distributed.run" in argv and argv[argv.index("--nproc-per-node") + 1] == "8"
    assert argv[argv.index("--master-addr") + 1] == "127.0.0.1" and argv[-6:] == ["--gpus", "8", "--steps", "2", "--warmup", "3"]
    # under torchrun (RANK set) it must not spawn again
    seen.clear()
    monkeypatch.setenv("RANK", "0")
    monkeypatch.setattr(bench, "run_ours", lambda args: seen.setdefault("ran", args.gpus))
    bench.main()
    assert seen == {"ran": 8}
