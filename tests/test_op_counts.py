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
    names = {("vl", "hlld"): "VL+PLM+HLLD (g=3)", ("vl", "roe"): "VL+PLM+Roe (g=3)", ("ctu", "hlld"): "CTU+PPM+HLLD char (g=4)",
             ("ctu", "roe"): "CTU+PPM+Roe char (g=4)"}
    # per-step counts: the 7 lines after each "<variant>, minimal ranges" line
    blocks = {}
    lines = out.splitlines()
    for n, ln in enumerate(lines):
        m = re.match(r"^(.*?), (maximal|minimal) ranges, per cell-update", ln)
        if m:
            blocks[(m.group(1), m.group(2))] = [int(re.search(r"flops per group\s+(\d+)", lines[n + 1 + q]).group(1)) for q in range(7)]
    for key, nm in names.items():
        assert vals[nm + ", maximal ranges, per cell-update"] == bench.FLOP_PER_CELL_UPDATE[key]["max"]
        assert vals[nm + ", minimal ranges, per cell-update"] == bench.FLOP_PER_CELL_UPDATE[key]["min"]
        assert blocks[(nm, "minimal")] == bench.FLOP_PER_GROUP_STEPS[key]
        # the steps add up to the whole update, and the minimal ranges never do more work than the maximal ones
        assert abs(sum(blocks[(nm, "minimal")]) / 16 ** 3 - bench.FLOP_PER_CELL_UPDATE[key]["min"]) < 0.06
        assert all(a <= b for a, b in zip(blocks[(nm, "minimal")], blocks[(nm, "maximal")]))
    # the solver hierarchy the paper names: HLLE < HLLD < Roe in work
    assert vals["per Riemann solve, HLLE"] < vals["per Riemann solve, HLLD"] < vals["per Riemann solve, Roe"]


def test_minimal_index_ranges_give_the_same_bits(oracle):
    """SURVEY Appendix B / DESIGN.md section 6: every stage evaluated only where the final update of the interior cells needs it
    (mhdref_config.minimal_ranges = 1, the ranges the kernels use) produces bitwise the outputs of the maximal ranges; the
    oracle's temporaries start as NaN, so a range cut one index too short would poison the result."""
    import numpy as np
    from paper_1804_03479_b200 import inputs
    for scheme, recon, g, N in ((0, 0, 3, 16), (0, 1, 4, 16), (1, 0, 3, 16), (1, 1, 4, 16), (1, 1, 4, 8), (0, 0, 4, 12)):
        U, B, dh = inputs.config2_batch(2, N=N, g=g)
        for riemann in (1, 2):
            a = oracle.advance(oracle.make_config(N=N, g=g, scheme=scheme, recon=recon, riemann=riemann), U, B, 2e-3, dh)
            b = oracle.advance(oracle.make_config(N=N, g=g, scheme=scheme, recon=recon, riemann=riemann, minimal_ranges=1), U, B, 2e-3, dh)
            for k in ("U", "B", "flux", "emf"):
                assert np.isfinite(b[k]).all() and np.array_equal(a[k], b[k]), (scheme, recon, g, N, riemann, k)
            assert all(x <= y for x, y in zip(b["stats"], a["stats"]))


def test_dram_traffic_table_is_readable_and_covers_the_default_line():
    """bench.py reads the ncu DRAM traffic of its roofline from profiles/r02_dram_traffic.csv at run time"""
    sys.path.insert(0, ROOT)
    import bench
    tr = bench.ncu_traffic()
    for prec in ("f32", "f64"):
        assert {"march_pass1", "march_pass2"} <= set(tr[("vl", "hlld", prec)]), tr.keys()
        for launches, mb in tr[("vl", "hlld", prec)].values():
            assert launches >= 1 and 10.0 < mb < 5000.0
