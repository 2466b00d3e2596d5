"""bench.py prints ONE JSON line with the keys the driver's contract names.  The reference arm (the CPU oracle on
host cores) is checked here without a GPU on the small config; the CUDA arm is checked on the GPU box."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BASE_KEYS = {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
             "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "cpu_baseline"}


def _run(*args, timeout=900):
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], cwd=ROOT, timeout=timeout,
                       stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1, lines
    return json.loads(lines[0])


def test_reference_arm_line():
    d = _run("--impl", "reference", "--workload", "cfg0", "--steps", "1", "--warmup", "0")
    assert BASE_KEYS <= set(d)
    assert d["impl"] == "reference" and d["dtype"] == "f64" and d["data"] == "synthetic"
    assert d["vs_baseline"] is None and d["higher_is_better"] is True
    assert d["value"] > 0 and d["unit"] == "interactions/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["cpu_baseline"]["cores"] >= 1 and d["cpu_baseline"]["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and "model" not in d["config"]


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       cwd=ROOT, env=env, timeout=300, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_cpu_baseline_sample_uses_every_thread():
    """The sampled oracle run is parallel over targets (not over the few sampled batches): its batch-sum phase scales
    with OMP_NUM_THREADS, and `cores` is the thread count the library really uses."""
    ncpu = os.cpu_count() or 1
    if ncpu < 4:
        pytest.skip("needs >= 4 cores")
    code = ("import bench, json; c = bench.workload('cfg0'); v, dt, desc, cores = bench.cpu_oracle_sample(c, repeat=2, n_batches=4); "
            "print(json.dumps({'dt': dt, 'cores': cores, 'value': v}))")
    res = {}
    for nt in (1, 4):
        env = dict(os.environ, OMP_NUM_THREADS=str(nt))
        r = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=env, timeout=600, stdout=subprocess.PIPE,
                           stderr=subprocess.PIPE, text=True)
        assert r.returncode == 0, r.stderr[-2000:]
        res[nt] = json.loads(r.stdout.strip().splitlines()[-1])
        assert res[nt]["cores"] == nt
    assert res[1]["dt"] / res[4]["dt"] > 2.0, res                # 4 threads: at least 2x faster than 1
    assert res[4]["value"] / res[1]["value"] > 2.0, res


@pytest.mark.gpu
def test_cuda_arm_line_small_workload():
    d = _run("--workload", "cfg0", "--steps", "3", "--warmup", "3")
    assert BASE_KEYS | {"roofline", "clocks", "phase_ms", "plan", "direct", "gi_update", "cpu_baseline_fast"} <= set(d)
    assert "impl" not in d or d["impl"] != "reference"
    assert d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] >= 3 and d["dtype"] == "f64"
    rf = d["roofline"]
    assert rf["bound"] == "alu" and rf["unit"] == "TFLOP/s" and 0.2 < rf["frac"] < 1.0
    assert abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert d["gpu_launches"] > 0
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == e["d2h_bytes_per_step"] == d["config"]["N"] * d["config"]["n_orb"] * 8
    assert e["value"] > 0 and e["value"] != d["value"] and e["bitwise_equal_to_device_path"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    assert d["cpu_baseline"]["cores"] == (os.cpu_count() if "OMP_NUM_THREADS" not in os.environ else int(os.environ["OMP_NUM_THREADS"]))
    ref = _run("--impl", "reference", "--workload", "cfg0", "--steps", "2", "--warmup", "1")
    assert ref["config"] == d["config"]                          # both arms describe the same workload
    assert 0.5 < ref["value"] / d["cpu_baseline"]["value"] < 2.0
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])
    assert abs(sum(d["phase_ms"].values()) - d["ms_per_step"]) < 0.2 * d["ms_per_step"]
