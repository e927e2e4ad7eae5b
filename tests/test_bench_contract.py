"""bench.py host logic without a GPU: the reference arm's JSON line (the oracle on the host cores,
same metric / unit / config keys), and the weak-scaling workload of rank r (disjoint point sets)."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--points", "64"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "interactions/s" and d["higher_is_better"] is True
    assert d["metric"].startswith("point-pixel DBIE interactions/sec") and d["dtype"] == "f64"
    assert d["value"] > 0 and d["steps"] == 1 and d["gpu_launches"] == 0 and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in d["config"] and "model" not in d["config"]


def test_rank_workloads_are_disjoint_and_equal_sized():
    sys.path.insert(0, ROOT)
    import bench
    a = bench.make_workload("cfg2", 0, 2)
    b = bench.make_workload("cfg2", 1, 2)
    assert a.M == b.M and np.array_equal(a.x, b.x) and np.array_equal(a.bz, b.bz)
    assert not np.intersect1d(a.z, b.z).size            # rank 1's layers are shifted by h/2
    s = bench.make_workload("cfg5")                     # config 5 defaults to a 16,384-point subset
    assert s.M == 16384 and (s.nx, s.ny) == (1024, 1024)
    assert bench.shard_info(100, 1, 4) == {"rank": 1, "world": 4, "points_per_rank": 100, "points_total": 400}


def test_fp64_instruction_counts_match_the_built_library():
    """bench.py's roofline multiplies interactions/s by the FP64-pipe instructions per interaction of each inner
    loop.  Those figures are recounted here from the SASS of the library as built (cuobjdump, no GPU needed)."""
    import importlib.util
    sys.path.insert(0, ROOT)
    import bench
    from paper_1306_1122_b200 import build as b
    b.build_lib()
    spec = importlib.util.spec_from_file_location("sass_loops", os.path.join(b.CSRC, "sass_loops.py"))
    sl = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(sl)
    table = dict(sl.loop_table(b.LIB, ("interact64_kernel", "solve_nm_fused_kernel")))

    def count(sub, which=0, per=1):
        (name, rows), = [(k, v) for k, v in table.items() if sub in k]
        r = rows[which]
        return r["pipes"]["fp64"] / (r["rsqrt"] * per)

    # kernel<MODE, NT, THREADS, MINB, UNR>: eval = mode 0 (loop 0: general lambda; loop 1: lambda = 0),
    # Eq. 13 stencil = mode 5 (loop 0: one sincos per component, kernel_n_near for the three offset positions), GRID NT = 8 = mode 2,
    # analytic gradient = mode 3, GRID on it (NT = 2) = mode 4
    assert count("interact64_kernel<(int)0, (int)1,") == bench.FP64_INSTR["eval"]
    assert count("interact64_kernel<(int)5, (int)1,") == bench.FP64_INSTR["nm"]
    assert count("solve_nm_fused_kernel<(int)5,") == bench.FP64_INSTR["nm"]
    assert count("interact64_kernel<(int)2, (int)8,", per=8) == bench.FP64_INSTR["grid"]
    assert count("interact64_kernel<(int)3, (int)1,") == bench.FP64_INSTR["analytic"]
    assert count("solve_nm_fused_kernel<(int)3,") == bench.FP64_INSTR["analytic"]
    assert count("interact64_kernel<(int)4, (int)2,", per=2) == bench.FP64_INSTR["grid_analytic"]
