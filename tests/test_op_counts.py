"""The algorithmic flop counts of bench.py's ALU roofline are the oracle's own: oracle/count_ops.cpp instantiates the
unchanged oracle with an operation-counting scalar.  This test rebuilds that tool and checks the constants in bench.py."""
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_bench_flop_constants_are_the_oracles_operation_counts(tmp_path):
    exe = str(tmp_path / "count_ops")
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-o", exe, os.path.join(ROOT, "oracle", "count_ops.cpp")])
    out = subprocess.check_output([exe], text=True)
    vals = {m.group(1).strip(): float(m.group(2)) for m in re.finditer(r"^(.*?)\s+flops\s+([0-9.]+)", out, flags=re.M)}
    sys.path.insert(0, ROOT)
    import bench
    assert vals["per Riemann solve, HLLD"] == bench.FLOP_PER_SOLVE["hlld"]
    assert vals["per Riemann solve, HLLE"] == bench.FLOP_PER_SOLVE["hlle"]
    assert vals["per Riemann solve, Roe"] == bench.FLOP_PER_SOLVE["roe"]
    assert vals["VL+PLM+HLLD (g=3), per cell-update"] == bench.FLOP_PER_CELL_UPDATE[("vl", "hlld")]
    assert vals["VL+PLM+Roe (g=3), per cell-update"] == bench.FLOP_PER_CELL_UPDATE[("vl", "roe")]
    assert vals["CTU+PPM+HLLD char (g=4), per cell-update"] == bench.FLOP_PER_CELL_UPDATE[("ctu", "hlld")]
    assert vals["CTU+PPM+Roe char (g=4), per cell-update"] == bench.FLOP_PER_CELL_UPDATE[("ctu", "roe")]
    # the solver hierarchy the paper names: HLLE < HLLD < Roe in work
    assert vals["per Riemann solve, HLLE"] < vals["per Riemann solve, HLLD"] < vals["per Riemann solve, Roe"]
