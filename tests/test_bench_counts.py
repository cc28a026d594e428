"""The operation counts bench.py prints beside the kernel's SASS count are the oracle's own ("an exact count
from the oracle, compiled with an operation-counting scalar type"), and the reference arm of bench.py describes the same
configuration as the GPU arm. CPU only."""
import json
import os
import subprocess
import sys

import bench
import orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_operation_counts_are_the_ones_bench_reports():
    (adds, muls, divs), bundle = orc.count_ops()
    assert adds + muls + divs == bench.ORACLE_ALGEBRA_OPS == 3576
    assert sum(bundle) == 188                                   # the oracle's own (unshared) bundle of one field
    assert bench.CANONICAL_DERIVATIVE_OPS == 2777
    assert bench.ORACLE_FLOP_PER_POINT_STAGE == 3576 + 2777
    # the credited count is the smaller one
    assert bench.ALG_FLOP_PER_POINT_STAGE <= bench.ORACLE_FLOP_PER_POINT_STAGE


def test_reference_arm_runs_the_whole_workload_and_names_the_same_config():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--n", "8",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, check=True, cwd=ROOT)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["gpu_launches"] == 0
    assert line["config"]["points"] == 8 ** 3 and line["config"]["workload"]
    assert "the whole of" in line["cpu_baseline"]["sample"] and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["value"] == line["value"] and line["e2e"]["h2d_bytes_per_step"] == 0
    w = bench.make_workload(0, 8)
    assert line["config"] == bench.config_of(w, 1)
