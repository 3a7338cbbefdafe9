"""bench.py's driver contract where it can be checked without a GPU: the reference arm (`--impl reference`, the CPU oracle
on a bounded sample) prints ONE JSON line with the keys the driver reads, under plain python and with the torchrun
environment of a non-zero rank (which must print nothing and exit 0); and the byte model that `roofline` is computed from
restates SURVEY.md 8(d)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(extra_env, *args):
    env = dict(os.environ, AXG_REFERENCE_BUDGET_S="2", **extra_env)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", *args], env=env,
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    return [ln for ln in r.stdout.splitlines() if ln.strip()]


def test_reference_arm_prints_the_contract_line():
    lines = _run({}, "--workload", "C1", "--gpus", "1", "--steps", "2", "--warmup", "1")
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"].startswith("particle-steps/s") and d["unit"] == "particle-steps/s"
    assert d["higher_is_better"] is True and d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 1
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None and d["data"] == "synthetic"
    assert d["config"]["workload"] == "C1" and "model" not in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] == 1 and cb["value"] == d["value"] and cb["sample"]
    e = d["e2e"]
    assert e["value"] == d["value"] and e["unit"] == d["unit"] and e["h2d_bytes_per_step"] == 0 == e["d2h_bytes_per_step"]


def test_reference_arm_is_silent_on_other_ranks():
    assert _run({"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"}, "--workload", "C1", "--gpus", "2") == []


def test_byte_model_restates_the_survey():
    sys.path.insert(0, ROOT)
    import bench
    from paper_1405_3331_b200 import workloads as W
    w = W.c3()
    n = 16_000_000
    step, own, launches, survey = bench.bytes_model(w, n, 0, 33, True)
    assert bench.key_passes(w.cells) == 3 and bench.key_passes(512 ** 3) == 3 and bench.key_passes(1024 * 1024 * 256) == 4
    assert survey["diffuse"] == 38.0 * n                                   # K1 = 17 read + 17 written + 4 key
    assert abs(step - ((38 + 44 + 42) * n + 8 * w.cells)) < 1e-6 * step    # + 3-pass sort 44, reorder 42, 8 B per cell
    assert own["diffuse"] == 45.0 * n and launches["diffuse"] == 1
    step_r, own_r, launches_r, survey_r = bench.bytes_model(w, n, 0, 33, False)
    assert step_r == step and launches_r["sort"] == 3 and own_r["diffuse"] == 38.0 * n
