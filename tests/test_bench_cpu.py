"""The parts of bench.py's contract that need no GPU: the reference arm (the oracle timed on the host cores,
`--impl reference`) prints one JSON line with the keys the driver reads; non-zero ranks of a torchrun launch do
nothing; `roofline.traffic` comes from the newest committed ncu capture; the CUDA arm refuses to run without a
device instead of falling back."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env=None):
    e = dict(os.environ)
    e.pop("RANK", None)
    e.pop("WORLD_SIZE", None)
    if env:
        e.update(env)
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True,
                          cwd=ROOT, env=e, timeout=600)


def test_reference_arm_prints_the_contract_line():
    r = _run(["--impl", "reference", "--workload", "C1", "--steps", "2", "--warmup", "1", "--reference-budget", "20"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "gauge_fix_iterations_per_s" and d["unit"] == "iterations/s"
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["value"] > 0 and d["steps"] >= 1 and d["ms_per_step"] > 0 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert abs(d["cpu_baseline"]["value"] - d["value"]) < 1e-12 and "sample" in d["cpu_baseline"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("C1: 8x8x8x8")


def test_reference_arm_other_ranks_exit_quietly():
    r = _run(["--impl", "reference", "--workload", "C1", "--steps", "1"], env={"RANK": "1", "WORLD_SIZE": "2"})
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_traffic_comes_from_the_newest_matching_capture():
    sys.path.insert(0, ROOT)
    import bench

    launched = {"update": ["k_sweep_tma<double, 3, 0, 1>"], "fft": ["k_fftr2_xy<double, 32, 0, 2, 0>", "k_fftr2_zt<double, 32, 32, 4>",
                                                                  "k_fftr2_xy<double, 32, 1, 4, 1>"]}
    caps, stale = bench.captured_traffic("C3", "fp64", 18, launched)
    up = caps["update"][0]
    assert up["bytes"] > 1.3e9 and up["kernel"].startswith("k_sweep_tma<double") and up["source"] == "profiles/r2c_traffic.csv"
    assert len(caps["fft"]) == 3 and all(r["bytes"] > 5e7 for r in caps["fft"])
    # a capture of a kernel this build does not launch is refused, not quoted
    caps2, stale2 = bench.captured_traffic("C3", "fp64", 18, {"update": ["k_sweep<double, 3, 3, 0, 0>"]})
    assert "update" not in caps2 and any("k_sweep_tma" in x for x in stale2)     # (refused: named under "stale")


def test_reduce_ncu_names_and_classes():
    sys.path.insert(0, ROOT)
    import bench

    n = bench.short_kernel_name("void lgf::k_sweep<double, (int)3, (bool)0, (bool)1, (int)3>(lgf::LinkPair<T1>, const lgf::C<T1> *)")
    assert n == "k_sweep<double, 3, 0, 1, 3>" and bench.kernel_class_of(n) == "update"
    assert bench.kernel_class_of("k_fftr2_zt<float, 32, 32, 4>") == "fft" and bench.kernel_class_of("k_finalize") is None


def test_cuda_arm_fails_loudly_without_a_device():
    import torch

    if torch.cuda.is_available():
        return                                    # on the GPU box the real thing is tested elsewhere
    r = _run(["--steps", "1", "--warmup", "1", "--no-variants", "--no-cpu-baseline", "--no-e2e"])
    assert r.returncode != 0 and "CUDA" in (r.stderr + r.stdout)
