"""bench.py end to end on a reduced workload: the JSON line carries the contract's keys, the rooflines are quoted
against ceilings measured in the same run, the host-facing leg was verified against the device-facing one, and the
oracle's FPR on the bounded sample equals the GPU's."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_line_on_a_reduced_workload():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--scale", "0.02", "--steps", "3", "--warmup", "3", "--read-batch", "50000",
           "--batches", "2", "--e2e-steps", "1", "--ref-insert-bases", "300000", "--ref-reads", "2000"]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "ceilings", "fpr"):
        assert key in line, key
    assert line["value"] > 0 and line["gpu_launches"] >= 3 * 4 and line["vs_baseline"] is None and line["dtype"] == "u64"
    assert line["config"]["workload"] == "config3" and line["n_gpus"] == 1 and line["steps"] == 3
    rf = line["roofline"]
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic", "traffic_source", "peak_source", "binds"):
        assert key in rf, key
    # quoted against the limit that binds the dominant kernel; the instruction roofline (both counts) and the step-level
    # fraction beside it
    assert rf["bound"] in ("alu", "hbm") and 0 < rf["frac"] < 1.5 and rf["peak_source"].startswith("measured")
    assert abs(rf["achieved"] / rf["peak"] - rf["frac"]) < 1e-9
    assert (rf["bound"] == "alu") == (rf["binds"] in ("alu_pipe", "fma_pipe", "issue"))
    assert 0 < rf["alu"]["frac"] < 1.5 and rf["alu"]["frac_with_survey_count"] > 0 and rf["alu"]["survey_ops_per_kmer"] in (63.0, 70.0)
    assert 0 < rf["step"]["frac"] < 1.2 and abs(rf["step"]["ms_per_step"] - line["ms_per_step"]) < 1e-9
    pipes = line["ceilings"]["pipe_warp_inst_per_clk_per_smsp"]
    assert 0.4 < pipes["LOP3"] < 0.6 and 0.4 < pipes["IMAD"] < 0.6 and 0.8 < pipes["LOP3:IMAD 1:1"] <= 1.05   # one per 2 clocks per pipe
    assert line["e2e"]["value"] > 0 and line["e2e"]["h2d_bytes_per_step"] > 0 and "verified" in line["e2e"]
    cb = line["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0
    ss = line["fpr"]["same_sample"]
    assert ss["hit_counts_identical"] and ss["gpu"] == ss["oracle"]
