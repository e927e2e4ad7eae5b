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


def _canned_full_record():
    """A full record of the shape measure_f64 + run_ours build (round 2's final default run, which printed
    21 KB on one line and overflowed the driver's stdout window), with this round's extra fields."""
    text = open(os.path.join(ROOT, "profiles", "r02_bench_default.json.txt")).read().strip().splitlines()[-1]
    full = json.loads(text)
    assert len(text) > 20000 and "legs" in full
    full["also"] = {k: {"value": v["value"], "ms_per_step": v["ms_per_step"], "frac": v["roofline"]["frac"]}
                    for k, v in full["legs"].items()}
    full["vs_previous_round"] = {"cfg4_eval": 1.0123456789, "cfg2_nm": 1.0456789123}
    full["cpu_baseline"]["cores_delivered"] = full["cpu_baseline"]["speedup_over_one_core"]
    full["config"]["sharding"] = "points, boundary replicated, no data-path collective"
    full["detail"] = "gpurun_out/bench_detail.json"
    return full


def test_headline_line_is_short_and_carries_the_contract_keys(capsys, tmp_path):
    """The driver parses the LAST stdout line and keeps about 3 KB of it: the line bench.py ends with must
    stay below 2,000 bytes whatever the full record holds, and carry every key of the contract."""
    sys.path.insert(0, ROOT)
    import bench
    full = _canned_full_record()
    text = bench.headline(full)
    assert len(text) < bench.HEADLINE_MAX_BYTES == 2000 and "\n" not in text
    d = json.loads(text)
    assert {"metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
            "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "roofline", "cpu_baseline",
            "gpu_launches"} <= set(d)
    assert "legs" not in d and not [k for k in d if k.endswith("_note")]
    assert d["value"] > 0 and d["unit"] == "interactions/s" and d["dtype"] == "f64" and d["vs_baseline"] is None
    assert {"workload", "boundary", "points", "step", "l2", "sharding"} <= set(d["config"]) and "model" not in d["config"]
    assert {"sm_mhz", "sm_max_mhz", "reasons"} <= set(d["clocks"])
    assert {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step", "api"} == set(d["e2e"])
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert {"bound", "kernel", "achieved", "peak", "unit", "frac", "frac_survey82", "frac_of_measured_dfma", "traffic",
            "kernel_ms_per_launch", "fp64_instr_per_interaction"} <= set(d["roofline"])
    assert abs(d["roofline"]["frac"] - d["roofline"]["achieved"] / d["roofline"]["peak"]) < 1e-4
    assert {"value", "unit", "cores", "cores_delivered", "kind", "sample"} == set(d["cpu_baseline"])
    assert not [k for k, v in d["roofline"].items() if isinstance(v, str) and len(v) > 60]
    assert set(d["also"]) == set(full["legs"]) and set(d["vs_previous_round"]) == {"cfg4_eval", "cfg2_nm"}
    # numbers keep 6 significant digits
    assert abs(d["value"] / full["value"] - 1.0) < 1e-5
    # a record that would not fit loses its optional parts, never the contract keys
    fat = dict(full, also={f"leg{i}": {"value": 1.0e11 + i, "ms_per_step": 1.5, "frac": 0.5} for i in range(40)})
    d2 = json.loads(bench.headline(fat))
    assert "also" not in d2 and "roofline" in d2 and len(bench.headline(fat)) < 2000
    # emit(): the full record goes to the detail file, the headline is the last (and only) stdout line
    path = tmp_path / "sub" / "detail.json"
    bench.emit(full, str(path))
    out = [l for l in capsys.readouterr().out.splitlines() if l.strip()]
    assert len(out) == 1 and json.loads(out[0])["detail"] == str(path) and len(out[0]) < 2000
    assert "legs" in json.load(open(path))


def test_traffic_table_names_its_captures():
    sys.path.insert(0, ROOT)
    import bench
    t = bench.ncu_traffic()
    assert {"eval", "nm", "f32"} <= set(t)
    for k, v in t.items():
        assert v["dram_bytes_per_launch"] > 0 and v["date"]
        assert os.path.exists(os.path.join(ROOT, v["capture"])), v["capture"]


def test_torchrun_relaunch_command_is_well_formed(monkeypatch):
    """`python bench.py --gpus N` outside torchrun re-launches itself with one rank per GPU on 127.0.0.1."""
    sys.path.insert(0, ROOT)
    import bench
    seen = {}
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: seen.setdefault("cmd", cmd) and 0)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "2", "--warmup", "3"])
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    try:
        bench.main()
    except SystemExit as e:
        assert e.code == 0
    cmd = seen["cmd"]
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nnodes=1" in cmd and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    i = cmd.index(os.path.join(ROOT, "bench.py"))
    assert cmd[i + 1:] == ["--gpus", "4", "--steps", "2", "--warmup", "3"]


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
    spec = importlib.util.spec_from_file_location("sass_loops", os.path.join(ROOT, "tests", "sass_loops.py"))
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
