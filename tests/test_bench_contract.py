"""-m "not gpu": bench.py's reference arm (the oracle on the host cores) prints the JSON line the contract asks for,
with the same `config` object the CUDA arm describes; the workload picker falls back when the box is too small."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    run = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600)
    assert run.returncode == 0, run.stderr[-2000:]
    return json.loads(run.stdout.strip().splitlines()[-1])


def test_reference_arm_prints_the_contract_line():
    line = _run("--impl", "reference", "--config", "4", "--records", "40000", "--steps", "2", "--warmup", "1")
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in line, key
    assert line["impl"] == "reference" and line["unit"] == "particles/s" and line["higher_is_better"] is True
    assert line["config"]["workload"] == "cfg4_psl_10x10" and line["config"]["records_per_gpu"] == 40000
    assert line["e2e"] == {"value": line["value"], "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] == 1 and line["gpu_launches"] == 0
    assert line["value"] > 1e5


def test_config_object_is_the_same_for_both_arms_and_the_picker_falls_back():
    sys.path.insert(0, ROOT)
    import argparse

    import bench
    import workloads as W

    w = W.config(5)
    a = bench.describe(w, 1, None)
    assert set(a) == {"workload", "baseline_config_index", "records_per_gpu", "record_bytes", "chunk_records", "keys", "mode",
                      "beams", "n_ebins", "position_bins", "sharding", "l2_policy"}
    assert a["workload"] == "cfg5_imrt_streamed" and a["records_per_gpu"] == 1_000_000_000 and a["beams"] == 9
    args = argparse.Namespace(config=0, records=0)
    idx, note = bench.pick_config(args, world=10 ** 6)  # a million ranks' worth of pinned memory: no box has it
    assert idx == 4 and "config 5 needs" in note
    assert bench.pick_config(argparse.Namespace(config=3, records=0), 1) == (3, None)
    # algorithmic bytes: the beam kernel reads 32-byte index records, writes SoA + key
    assert bench.algorithmic_bytes("beam", 0, 0, 1000, 100, False) == 32 * 1000 + 36 * 100
    assert bench.algorithmic_bytes("count_keys", 0, 500, 0, 0, False) == 4 * 500
