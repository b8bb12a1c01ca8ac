"""The JSON line `bench.py` prints (the driver's contract), checked on the committed lines of the final code under
profiles/ -- no GPU needed: every key the contract names is present and self-consistent."""
import json
import os

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def load(name):
    with open(os.path.join(ROOT, "profiles", name)) as f:
        return [json.loads(l) for l in f if l.startswith("{")]


def check_line(d, reference=False):
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "e2e", "cpu_baseline"):
        assert k in d, k
    assert d["higher_is_better"] is True and d["vs_baseline"] is None and d["data"] == "synthetic" and d["dtype"] == "f32"
    assert d["unit"] == "evals/s" and "workload" in d["config"] and "model" not in d["config"]
    e = d["e2e"]
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in e, k
    if reference:
        assert d["impl"] == "reference" and e["h2d_bytes_per_step"] == 0 and e["value"] == d["value"]
        cb = d["cpu_baseline"]
        assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
        return
    assert d["warmup"] >= 3 and d["gpu_launches"] > 0
    assert e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0 and 0 < e["value"] <= d["value"] * 1.02
    c = d["clocks"]
    if d["ms_per_step"] * d["steps"] > 400:      # the sampler's period is 200 ms (C1 and C2 finish sooner)
        assert c["sm_mhz"] <= c["sm_max_mhz"]
    assert not [r for r in c["reasons"] if "slowdown" in r]
    r = d["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in r, k
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    # value = evaluations of the timed steps / device time
    ev = d["config"]["evaluations_per_step"]
    assert abs(d["value"] - ev / (d["ms_per_step"] * 1e-3)) <= 1e-6 * d["value"]


def test_headline_line_c5():
    (d,) = load("r3_bench_c5.json.txt")
    check_line(d)
    assert d["config"]["workload"].startswith("C5: fixed 260x311x260") and d["config"]["transforms"] == 68921
    r = d["roofline"]
    assert r["bound"] == "shared-atomic" and r["frac"] >= 0.5            # north_star's target on this map
    assert r["traffic"] is not None and r["traffic"] > r["algorithmic_bytes_per_step"]
    # frac counts the updates issued, not the evaluations; the probed peak is the larger of the two random-bin probes
    assert r["frac"] == r["frac_issued"] <= r["frac_by_evaluations"] and r["peak_round1_pattern"] > r["peak"]
    assert r["updates_issued_per_step"] <= d["config"]["evaluations_per_step"]
    assert abs(r["achieved"] - r["updates_issued_per_step"] / (r["kernel_ms_per_step"] * 1e-3) / 1e9) <= 1e-6 * r["achieved"]
    assert r["peak"] == max(r["peak_probe_hash_in_loop"], r["peak_probe_hash_hoisted"])
    assert r["peak"] <= r["peak_nominal"] and abs(r["frac_of_nominal"] - r["achieved"] / r["peak_nominal"]) < 1e-9
    assert r["kernel_ms_per_step"] <= d["ms_per_step"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and 0 < cb["value"] < d["value"]


def test_rotation_line_c3_is_measured_against_a_hardware_floor():
    (d,) = load("r3_bench_c3.json.txt")
    check_line(d)
    r = d["roofline"]
    assert d["config"]["workload"].startswith("C3") and r["bound"] == "l1tex-writeback"
    assert 0 < r["frac"] < 1 and abs(r["clocks_per_warp_sample"] - 20.41) < 1e-9
    # the kernel without its updates is a diagnostic beside the line, not its peak
    assert r["same_kernel_without_updates"]["rate"] < r["peak"] and "peak_gathers_plus_updates" not in r


def test_all_configs_from_one_invocation():
    lines = load("r3_bench_all.json.txt")
    assert [l["config"]["workload"][:2] for l in lines] == ["C1", "C2", "C3", "C4", "C5"]   # the headline last
    for d in lines:
        d = dict(d, cpu_baseline=d.get("cpu_baseline"))
        check_line(d)


def test_reference_arm_line():
    (d,) = load("r3_bench_reference.json.txt")
    check_line(d, reference=True)
    (ours,) = load("r3_bench_c5.json.txt")
    assert d["config"]["workload"] == ours["config"]["workload"] and d["metric"] == ours["metric"]
