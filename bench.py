#!/usr/bin/env python
"""bench.py — throughput of the DBIE hot path on B200 (one process per GPU).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg4|cfg2|cfg3|cfg5] [--method nm|grid] [--gradient fd|analytic]
                    [--dtype f64|f32] [--points P] [--slabs] [--legs] [--detail FILE]

The metric is BASELINE.json's: point-pixel DBIE interactions/s in fp64 and the fraction of the FP64
roofline.  One interaction = one (evaluation point, pixel) pair, all three components; in the solver
every stencil position and every objective evaluation counts.

Default (no flags, one GPU): the HEADLINE line is BASELINE configs[3] ("cfg4": 512x512 boundary,
M = 1,048,576 random points, per-component lambda, fp64) — the configuration the metric's "interactions/s
and roofline fraction" are quoted on.  A step is one pass of the hot path over that batch: stage the
boundary (dbie_create) and evaluate Eq. 6/16 at every point (dbie_eval).  The same run also times BASELINE
configs[1] ("cfg2": the full per-point Nelder-Mead solve of the 64x64x32 Low & Lou volume) for two steps and
reports it under "also", so that both workloads stay comparable from round to round ("vs_previous_round").
`value` is measured with the inputs resident in HBM; `e2e` goes through the host-pointer C-ABI calls with
the copies inside the timed region.  `roofline` is for the dominant kernel, timed live with CUDA-event pairs
around each of its launches.  `cpu_baseline` times the oracle, as it stands, on the host cores (all cores and
one core) over a bounded sample.

Output: the LAST line of stdout (rank 0) is ONE compact JSON line of fewer than 2,000 bytes (`headline`): the
contract keys only, no prose.  What each field means is in DESIGN.md section 7.  `--detail FILE` also writes the
full record (every diagnostic field, the pass timeline, the operand probe) to FILE; `--legs` times four more
legs (48-point latency, config 5 GRID, fp32, reduced sincos) and puts their full records into that file
(default gpurun_out/bench_detail.json when --legs is given) and their values into "also".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "point-pixel DBIE interactions/sec (fp64)"
UNIT = "interactions/s"
# FP64-pipe instructions per interaction of each inner loop, counted from the SASS of the built library by
# tests/sass_loops.py (profiles/r02_sass_loops.txt); DESIGN.md section 6 derives them.
FP64_INSTR = {"eval": 61.0, "eval_reduced": 55.0, "nm": 418 / 8, "analytic": 86.0, "grid": 200 / 8, "grid_analytic": 158 / 2}
FP64_INSTR_SURVEY = 82               # SURVEY.md 8(d) canonical count
SM_COUNT, FP64_LANES_PER_SM = 148, 64   # B200: 148 SMs, 64 FP64 lanes per SM per clock
MUFU_PER_INTERACTION = 7             # dbie_eval_f32 default (SFU sincos): 1 rsqrt + 3 x (sin, cos)
MUFU_LANES_PER_SM = 16

# Results of the previous round's final runs (profiles/r02_bench_default.json.txt, r02_bench_cfg2_solve.json.txt):
# the default line reports this round's value over these, workload by workload.
PREVIOUS_ROUND = {"cfg4_eval": 2.56e11, "cfg2_nm": 2.79e11}
HEADLINE_MAX_BYTES = 2000            # the driver keeps about 3 KB of stdout: the last line must fit with room to spare


def ncu_traffic() -> dict:
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of ONE launch of the dominant kernel, from the
    committed `ncu --set full` captures named in profiles/traffic.json (kind -> bytes, capture file, date), so
    that a stale figure is visible next to its source; evidence that HBM is idle (the bound is the FP64 pipe)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return json.load(f)["kernels"]
    except (OSError, ValueError, KeyError):
        return {}


def make_workload(name: str, rank: int = 0, world: int = 1, points: int = 0):
    """The rank's batch.  Weak scaling: every rank gets a batch of the same size; rank r's points are
    shifted by r*h/world in z so the ranks' point sets are disjoint.  `points` > 0 takes a seeded subset."""
    import workloads
    wl = {"cfg2": workloads.config2, "cfg3": workloads.config3, "cfg4": workloads.config4,
          "cfg5": workloads.config5}[name]()
    if points <= 0 and name == "cfg5":
        points = 16384    # the full 8.4e6-point GRID solve is 2.8e15 interactions: hours at the roofline
    if 0 < points < wl.M:
        wl, _ = wl.seeded_subset(points, seed_offset=900)
    if world > 1:
        wl.z = wl.z + rank * wl.h / world
    return wl


SHARDING = "points, boundary replicated, no data-path collective"


def shard_info(M: int, rank: int, world: int) -> dict:
    """Points are independent: no data-path collective, results stay on the rank."""
    return {"rank": rank, "world": world, "points_per_rank": M, "points_total": M * world}


def reduce_over_ranks(dist, device, ms: float, interactions: float):
    """max over ranks of the time, sum over ranks of the work (the contract's aggregate)."""
    from paper_1306_1122_b200 import sharding
    return sharding.reduce_over_ranks(dist, device, ms, interactions)


class ClockSampler:
    """nvidia-smi clocks line of B200_PROFILING.md, sampled during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
                for n, v in zip(names, r[5:9]):
                    if v.strip().lower() == "active":
                        reasons.add(n)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        hi = [s for s, p in zip(sm, pw) if p >= 0.6 * max(pw)] or sm     # samples under load
        return {"sm_mhz": float(np.median(hi)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


class Mode:
    """What a leg runs: eval at given lambda, or the lambda solve (NM / GRID, Eq. 13 / analytic gradient)."""

    def __init__(self, workload: str, grid: bool = False, analytic: bool = False, points: int = 0,
                 reduced: bool = False):
        self.workload, self.grid, self.analytic, self.points = workload, grid, analytic, points
        self.reduced = reduced          # eval only: DBIE_EVAL_REDUCED_SINCOS (reading A-12)

    def kind(self, is_solve: bool) -> str:
        if not is_solve:
            return "eval_reduced" if self.reduced else "eval"
        if self.grid:
            return "grid_analytic" if self.analytic else "grid"
        return "analytic" if self.analytic else "nm"


# --------------------------------------------------------------------------- oracle legs ---
def oracle_timed(wl, mode: Mode, npoints: int, seed_offset: int, nthreads: int = 0) -> dict:
    """Time the oracle's solve (or eval) on a seeded sample of the workload's points."""
    import oracle
    sub, _ = wl.seeded_subset(npoints, seed_offset=seed_offset)
    t0 = time.perf_counter()
    if wl.lam is None and mode.grid:
        o = oracle.Opts(method=1, analytic=1 if mode.analytic else 0)
        out = oracle.solve_grid(sub, o, nthreads=nthreads)
        inter = float(out["iters"].sum()) * o.n_trial * (1.0 if o.analytic else 4.0) * wl.N
    elif wl.lam is None:
        an = 1 if mode.analytic else 0
        out = oracle.solve_nm(sub, oracle.Opts(analytic=an), nthreads=nthreads)
        inter = float(out["nfev"].sum()) * (1.0 if an else 4.0) * wl.N
    else:
        oracle.eval(sub, nthreads=nthreads)
        inter = float(sub.M) * wl.N
    dt = time.perf_counter() - t0
    return {"seconds": dt, "interactions": inter, "points": sub.M}


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(wl, mode: Mode, target_s: float = 15.0) -> dict:
    """Oracle as it stands on the host cores (all cores AND one core).  A one-core probe
    sizes the samples: ~target_s of wall time on all cores, about a third of that on one core."""
    import oracle
    cores = oracle.max_threads()
    # one core first: a small probe gives the core-seconds per point, which sizes both samples
    r1 = oracle_timed(wl, mode, min(wl.M, 1 if wl.lam is None else 8), seed_offset=52, nthreads=1)
    per_point_core = r1["seconds"] / max(r1["points"], 1)
    if r1["seconds"] < 0.5 * target_s / 3.0:
        n1 = int(min(wl.M, max(1, (target_s / 3.0) / max(per_point_core, 1e-9))))
        r1 = oracle_timed(wl, mode, n1, seed_offset=53, nthreads=1)
        per_point_core = r1["seconds"] / max(r1["points"], 1)
    # all cores: a probe (a few scheduling chunks per core) measures the parallel rate actually delivered
    # (a container may expose more cores than its CPU quota), then the sample is sized from it
    r = oracle_timed(wl, mode, min(wl.M, cores * (1 if wl.lam is None else 16)), seed_offset=50)
    if r["seconds"] < 0.5 * target_s:
        n = int(min(wl.M, 65536, max(cores, target_s * r["points"] / max(r["seconds"], 1e-9))))
        r = oracle_timed(wl, mode, n, seed_offset=51)
    kind = ("solve_grid" if mode.grid else "solve_nm") if wl.lam is None else "eval"
    return {"value": r["interactions"] / r["seconds"], "unit": UNIT, "cores": cores, "kind": "oracle",
            "cpu": cpu_model(),
            "sample": f"oracle.{kind} on {r['points']} seeded points of {wl.name} "
                      f"({r['interactions']:.3e} interactions in {r['seconds']:.1f} s)",
            "cores_delivered": (r["interactions"] / r["seconds"]) / (r1["interactions"] / r1["seconds"]),
            "speedup_over_one_core": (r["interactions"] / r["seconds"]) / (r1["interactions"] / r1["seconds"]),
            "speedup_note": "all-threads rate / one-thread rate: well below `cores` when the box exposes more cores than "
                            "its CPU quota delivers",
            "one_core": {"value": r1["interactions"] / r1["seconds"], "cores": 1,
                         "sample": f"{r1['points']} points ({r1['interactions']:.3e} interactions in {r1['seconds']:.1f} s)"}}


def run_reference(args, mode: Mode) -> None:
    """--impl reference: the oracle timed on the host cores, same metric / config / unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    wl = make_workload(mode.workload, points=mode.points)
    cores = oracle.max_threads()
    probe = oracle_timed(wl, mode, min(wl.M, cores), seed_offset=60)
    per_point = probe["seconds"] / probe["points"]
    budget = 150.0 / max(args.steps + args.warmup, 1)            # whole run within a few minutes
    n = int(min(wl.M, max(cores, min(budget, 20.0) / per_point)))
    for w in range(args.warmup):
        oracle_timed(wl, mode, n, seed_offset=100 + w)
    tot_s = tot_i = 0.0
    for k in range(args.steps):
        r = oracle_timed(wl, mode, n, seed_offset=200 + k)
        tot_s += r["seconds"]; tot_i += r["interactions"]
    value = tot_i / tot_s
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "gpu_launches": 0,
        "config": workload_config(wl, mode, n_points_per_step=n),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model(),
                         "sample": f"each step: oracle on {n} seeded points of {wl.name}"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    line["cpu_baseline"]["value"] = line["e2e"]["value"] = _sig(value)   # the line's own value, digit for digit
    print(headline(line), flush=True)


def workload_config(wl, mode: Mode, n_points_per_step=None) -> dict:
    desc = {"cfg2": "BASELINE configs[1]: Low&Lou n=1 m=1 l=0.3 Phi=pi/4, boundary 64x64 on [-1,1]^2, "
                    "full per-point lambda solve on the 64x64x32 volume",
            "cfg3": "BASELINE configs[2]: synthetic bipolar AR 256x256 at 0.5 Mm/px, lambda solve on 128x128x64",
            "cfg4": "BASELINE configs[3]: eval at fixed lambda, boundary 512x512, M=1,048,576 random points, "
                    "per-component lambda in [-0.2,0.2]/px",
            "cfg5": "BASELINE configs[4]: quadrupolar delta-spot 1024x1024, lambda solve on a seeded subset of "
                    "the 256x256x128 volume"}[mode.workload]
    if getattr(mode, "reduced", False):
        desc += " [DBIE_EVAL_REDUCED_SINCOS: eval-only reduced-degree sincos, reading A-12; max |dB|/|B| 2e-12 vs the oracle]"
    if wl.lam is None:
        desc += " [method: " + ("GRID T=8, 10 levels" if mode.grid else "Nelder-Mead") + (
            "; analytic gradient (O-5): 1 evaluation position per objective evaluation instead of 4"
            if mode.analytic else "") + "]"
    return {"workload": desc, "boundary": [wl.nx, wl.ny], "points": wl.M if n_points_per_step is None
            else n_points_per_step, "step": "dbie_create + dbie_solve" if wl.lam is None else "dbie_create + dbie_eval",
            "l2": "flushed between timed steps (256 MiB write)"}


# --------------------------------------------------------------------------- the line ------
def _sig(v, digits=6):
    """Floats to `digits` significant digits (the line is read by a parser with a 3 KB window)."""
    if isinstance(v, float):
        return float(f"{v:.{digits}g}")
    if isinstance(v, dict):
        return {k: _sig(x, digits) for k, x in v.items()}
    if isinstance(v, (list, tuple)):
        return [_sig(x, digits) for x in v]
    return v


def _pick(d, keys):
    return None if d is None else {k: d[k] for k in keys if k in d}


HEADLINE_KEYS = ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                 "scaling", "vs_baseline", "dtype", "data", "gpu_launches")
HEADLINE_SUB = {
    "config": ("workload", "boundary", "points", "step", "l2", "sharding", "points_total"),
    "clocks": ("sm_mhz", "sm_max_mhz", "power_w_max", "reasons"),
    "e2e": ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step", "api"),
    "roofline": ("bound", "kernel", "achieved", "peak", "unit", "frac", "frac_survey82", "frac_of_measured_dfma",
                 "traffic", "kernel_ms_per_launch", "kernel_share_of_step", "fp64_instr_per_interaction",
                 "mufu_per_interaction"),
    "cpu_baseline": ("value", "unit", "cores", "cores_delivered", "kind", "sample"),
}


def headline(full: dict) -> str:
    """The ONE line bench.py ends with: the contract keys of `full`, numbers at 6 significant digits, no prose
    (field meanings: DESIGN.md section 7).  Always shorter than HEADLINE_MAX_BYTES: optional parts are dropped,
    least important first, if a record would not fit (it does not happen with the records this file builds;
    tests/test_bench_contract.py pins the size on canned numbers)."""
    line = {k: full[k] for k in HEADLINE_KEYS if k in full}
    for name, keys in HEADLINE_SUB.items():
        if name in full:
            line[name] = _pick(full[name], keys)
    for k in ("also", "vs_previous_round", "detail"):
        if full.get(k) is not None:
            line[k] = full[k]
    line = _sig(line)
    for drop in (None, "detail", "also", "vs_previous_round"):
        if drop:
            line.pop(drop, None)
        text = json.dumps(line, separators=(",", ":"))
        if len(text) < HEADLINE_MAX_BYTES:
            return text
    raise RuntimeError(f"bench.py: the headline line has {len(text)} bytes (limit {HEADLINE_MAX_BYTES})")


def emit(full: dict, detail_path: str = "") -> None:
    """Write the full record to `detail_path` (if given), then print the headline as the last stdout line."""
    if detail_path:
        try:
            os.makedirs(os.path.dirname(os.path.abspath(detail_path)), exist_ok=True)
            with open(detail_path, "w") as f:
                json.dump(full, f, indent=1)
            full = dict(full, detail=detail_path)
        except OSError as e:
            print(f"bench.py: could not write {detail_path}: {e}", file=sys.stderr)
    print(headline(full), flush=True)


# --------------------------------------------------------------------------- our arm -------
def measure_f64(mode: Mode, steps: int, warmup: int, rank=0, world=1, local=0, dist=None, e2e: bool = True) -> dict:
    """Time `steps` passes of dbie_create + dbie_eval / dbie_solve on this rank's batch; returns the line."""
    import torch
    import paper_1306_1122_b200 as dbie
    dev = torch.device("cuda", local)
    wl = make_workload(mode.workload, rank, world, points=mode.points)
    is_solve = wl.lam is None
    kind = mode.kind(is_solve)
    sopts = dbie.default_opts(method=1 if mode.grid else 0, analytic=1 if mode.analytic else 0)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(dev)
    d_bx, d_by, d_bz = t(wl.bx), t(wl.by), t(wl.bz)
    d_x, d_y, d_z = t(wl.x), t(wl.y), t(wl.z)
    d_lam = None if is_solve else t(wl.lam)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device(profile=False):
        ctx = dbie.DBIE(wl.nx, wl.ny, wl.h, wl.x0, wl.y0, d_bx, d_by, d_bz, reduced_sincos=mode.reduced)
        if profile:
            ctx.profile(True)
        out = ctx.solve(d_x, d_y, d_z, sopts) if is_solve else ctx.eval(d_x, d_y, d_z, d_lam)
        return ctx, out

    # e2e inputs live in pinned host memory (numpy views of pinned tensors keep them alive)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).pin_memory()
    _pinned = {k: pin(getattr(wl, k)) for k in ("bx", "by", "bz", "x", "y", "z")}
    if not is_solve:
        _pinned["lam"] = pin(wl.lam)
    hp = {k: v.numpy() for k, v in _pinned.items()}

    def step_host():
        ctx = dbie.DBIE(wl.nx, wl.ny, wl.h, wl.x0, wl.y0, hp["bx"], hp["by"], hp["bz"], reduced_sincos=mode.reduced)
        out = (ctx.solve_host(hp["x"], hp["y"], hp["z"], sopts) if is_solve
               else ctx.eval_host(hp["x"], hp["y"], hp["z"], hp["lam"]))
        return ctx, out

    for _ in range(max(warmup, 0)):
        ctx, _ = step_device()
        torch.cuda.synchronize()
        ctx.close()

    # ---- timed: K steps, device-resident inputs, CUDA events on the launching stream
    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    ms_total = inter_total = kern_ms = 0.0
    launches = kern_launches = evals = 0
    pass_trace = None
    for k in range(steps):
        flush_buf.zero_()                       # L2 flush, outside the event pair
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx, out = step_device(profile=True)
        e1.record()
        e1.synchronize()
        ms_total += e0.elapsed_time(e1)
        c = ctx.counters()
        kt = ctx.kernel_time()
        inter_total += c["interactions"]
        launches += c["launches"] + 1           # + the boundary staging kernel
        evals += c["objective_evals"]
        kern_ms += kt["interact_ms"]
        kern_launches += kt["interact_launches"]
        if is_solve and not mode.grid and k == steps - 1:
            pass_trace = ctx.pass_trace()
        ctx.close()
    barrier()
    clocks = sampler.stop() if sampler else None
    ms_max, inter_sum = reduce_over_ranks(dist, dev, ms_total, inter_total)
    value = inter_sum / (ms_max * 1e-3)

    # ---- e2e: host buffers through the _host C-ABI calls, copies inside the timed region
    e2e_line = None
    if e2e:
        ctx, _ = step_host(); ctx.close()
        barrier()
        t0 = time.perf_counter()
        e2e_inter = 0.0
        step_ms = []
        for k in range(steps):
            ts = time.perf_counter()
            ctx, out = step_host()
            e2e_inter += ctx.counters()["interactions"]
            ctx.close()
            step_ms.append((time.perf_counter() - ts) * 1e3)
        torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) * 1e3
        barrier()
        e2e_ms, e2e_inter = reduce_over_ranks(dist, dev, e2e_ms, e2e_inter)
        h2d = 3 * wl.N * 8 + 3 * wl.M * 8 + (0 if is_solve else 3 * wl.M * 8)
        d2h = (3 + 3 + 2) * wl.M * 8 + 2 * wl.M * 4 if is_solve else 3 * wl.M * 8
        e2e_line = {"value": e2e_inter / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / steps,
                    "ms_each_step": [round(t, 3) for t in step_ms],
                    "ms_each_step_note": "host wall clock of every timed step on this rank (create, copies, kernels, "
                                         "destroy); `value` uses their sum: a spread between steps is host-side jitter "
                                         "(cudaMalloc/cudaFree, page faults of the output buffer) on a shared box",
                    "api": "dbie_create_host + dbie_solve_host" if is_solve else "dbie_create_host + dbie_eval_host"}
    if rank != 0:
        return {}

    # ---- roofline of the dominant kernel, FP64-pipe bound
    try:
        dfma_meas, ffma_meas = dbie.probe_dfma_rate(300.0)
    except Exception:
        dfma_meas = ffma_meas = None
    try:
        operand_probe = dbie.probe_fp64_operands(100.0) if not is_solve else None   # eval legs only
    except Exception:
        operand_probe = None
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak_slots = SM_COUNT * FP64_LANES_PER_SM * sm_max * 1e6          # FP64 lane-instructions / s
    kern_ips = inter_total / (kern_ms * 1e-3) if kern_ms > 0 else 0.0
    per_inter = FP64_INSTR[kind]
    achieved_slots = kern_ips * per_inter
    traffic = ncu_traffic().get(kind) if (mode.points == 0 and not mode.reduced and
                                          mode.workload == ("cfg4" if not is_solve else "cfg2")) else None
    traffic = (traffic["dram_bytes_per_launch"], f"{traffic['capture']} ({traffic['date']})") if traffic else None
    kernel_name = "dbie::interact64_kernel" if (not is_solve or mode.grid) else "dbie::solve_nm_fused_kernel"
    kernel_what = ("fp64 point-pixel sums" if (not is_solve or mode.grid) else
                   "whole Nelder-Mead search in one cooperative launch: point-pixel sums + residual + simplex step + "
                   "list compaction")
    # independent-geometry rate: objective evaluations x N, without the x4 stencil or xT trial multipliers
    pos = 1.0 if (not is_solve or mode.analytic) else 4.0
    indep = (inter_total / pos / (8.0 if mode.grid else 1.0)) / (ms_total * 1e-3)
    roofline = {
        "bound": "alu", "kernel": kernel_name, "kernel_what": kernel_what,
        "achieved": 2e-12 * achieved_slots, "peak": 2e-12 * peak_slots, "unit": "TFLOP/s",
        "frac": achieved_slots / peak_slots,
        "unit_note": "achieved and peak count every FP64-pipe lane-instruction (DFMA, DMUL, DADD alike) as 2 flop: "
                     "`frac` is the fraction of the FP64 pipe's issue slots, not of real flops",
        "achieved_lane_instr_per_s": achieved_slots, "peak_lane_instr_per_s": peak_slots,
        "traffic": traffic[0] if traffic else None,
        "traffic_source": traffic[1] if traffic else "no ncu --set full capture of this leg at this size; see profiles/README.md",
        "traffic_note": "DRAM bytes of one launch.  Algorithmic bytes: eval 72 M + 32 N (cfg4: 84 MB); solve: 24 M of "
                        "point data + 480 M of optimiser state per pass through L2.  HBM is idle either way (bound: FP64 pipe)",
        "note": "FP64-pipe bound (no HBM/tensor step): achieved = interactions/s of the kernel x FP64 lane-instructions per "
                "interaction (eval 61, 55 with DBIE_EVAL_REDUCED_SINCOS; Eq. 13 stencil 52.25; GRID T=8 25; analytic gradient 86; GRID on it 79; "
                "profiles/r02_sass_loops.txt) x 2; peak = 148 SM x 64 FP64 lanes x clocks.max.sm (derived, DESIGN.md s7)",
        "kernel_interactions_per_s": kern_ips, "kernel_ms_per_launch": kern_ms / max(kern_launches, 1),
        "kernel_launches": kern_launches, "kernel_share_of_step": kern_ms / ms_total if ms_total else None,
        "fp64_instr_per_interaction": per_inter,
        "frac_survey82": kern_ips * FP64_INSTR_SURVEY / peak_slots,
        "frac_survey82_note": "SURVEY 8(d)'s canonical 82 instructions per interaction; exceeds `frac` (and can exceed 1) "
                              "where the kernel executes fewer: the stencil positions / GRID trials share sincos work",
        "peak_measured_dfma_per_s": dfma_meas, "peak_measured_ffma_per_s": ffma_meas,
        "frac_of_measured_dfma": (achieved_slots / dfma_meas) if dfma_meas else None,
    }
    if pass_trace is not None and pass_trace["npass"] > 0:
        # the pass timeline of the last timed solve (dbie_last_pass_trace): where the fused kernel's time goes
        act, pms = pass_trace["active"].astype(np.float64), pass_trace["ms"]
        per_eval = (1.0 if mode.analytic else 4.0) * wl.N
        bins = []
        grid_pts = SM_COUNT * 2 * 128                      # one round of the persistent grid: 296 CTAs x 128 points
        for lo, hi, label in ((0, 512, "<= 512"), (512, 4096, "513 - 4,096"), (4096, grid_pts // 2, "4,097 - half a round"),
                              (grid_pts // 2, grid_pts, "half a round - one round (37,888)"),
                              (grid_pts, 2 * grid_pts, "one - two rounds"), (2 * grid_pts, 1e18, "> two rounds")):
            m = (act > lo) & (act <= hi)
            if m.any():
                bins.append({"active_points": label, "passes": int(m.sum()), "ms": float(pms[m].sum()),
                             "interactions_per_s": float(act[m].sum() * per_eval / (pms[m].sum() * 1e-3))})
        roofline["passes"] = {"count": int(pass_trace["npass"]), "ms_total": float(pms.sum()), "by_active_points": bins,
                              "note": "one pass = one objective evaluation of every still-active point, ended by a grid-wide "
                                      "barrier; a work item cannot be smaller than one canonical chunk of 128 points, so passes "
                                      "that fill less than a round of the 296 CTAs run below the inner loop's rate"}
    if operand_probe:
        roofline["fp64_operand_probe_per_s"] = operand_probe
        roofline["fp64_operand_probe_note"] = (
            "lane-instructions/s of register-only loops: a DFMA that reads three different registers issues every 3 "
            "cycles instead of 2 (DESIGN.md section 6), so the FP64-pipe peak is not reachable by a loop that needs them")
    return {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": warmup, "ms_per_step": ms_max / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": dict(workload_config(wl, mode), **shard_info(wl.M, rank, world), sharding=SHARDING,
                       objective_evals_per_step=evals / steps),
        "clocks": clocks,
        "e2e": e2e_line,
        "gpu_launches": launches,
        "independent_geometry_interactions_per_s": indep,
        "independent_geometry_note": "objective evaluations (or eval points) x pixels per second: without the x4 stencil "
                                     "positions of Eq. 13 and the x8 GRID trials that `value` counts as interactions",
        "roofline": roofline,
    }


def measure_f32(steps: int, warmup: int, points: int = 0) -> dict:
    """BASELINE configs[3] "fp64 and fp32": dbie_eval_f32 on the config-4 workload (one GPU).
    Same JSON contract; the roofline is the SFU (MUFU sin/cos of the reduced argument, 7 per interaction)."""
    import torch
    import paper_1306_1122_b200 as dbie
    dev = torch.device("cuda", 0)
    wl = make_workload("cfg4", points=points)
    t64 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(dev)
    h32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).pin_memory()
    d_bx, d_by, d_bz = t64(wl.bx), t64(wl.by), t64(wl.bz)
    hx, hy, hz, hl = h32(wl.x), h32(wl.y), h32(wl.z), h32(wl.lam)
    dx, dy, dz, dl = hx.to(dev), hy.to(dev), hz.to(dev), hl.to(dev)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    inter = float(wl.M) * wl.N

    def step(profile=False):
        ctx = dbie.DBIE(wl.nx, wl.ny, wl.h, wl.x0, wl.y0, d_bx, d_by, d_bz, fp32=True)
        if profile:
            ctx.profile(True)
        return ctx, ctx.eval_f32(dx, dy, dz, dl)

    for _ in range(max(warmup, 0)):
        ctx, _ = step(); torch.cuda.synchronize(); ctx.close()
    sampler = ClockSampler(0)
    torch.cuda.synchronize()
    ms_total = kern_ms = 0.0
    kern_launches = launches = 0
    for k in range(steps):
        flush_buf.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx, out = step(profile=True)
        e1.record(); e1.synchronize()
        ms_total += e0.elapsed_time(e1)
        kt = ctx.kernel_time()
        kern_ms += kt["interact_ms"]; kern_launches += kt["interact_launches"]
        launches += ctx.counters()["launches"] + 1
        ctx.close()
    clocks = sampler.stop()
    # e2e: host boundary and pinned host float32 points through the _host C-ABI calls, float32 B back out, every step
    hb = wl.bx, wl.by, wl.bz
    hxn, hyn, hzn, hln = hx.numpy(), hy.numpy(), hz.numpy(), hl.numpy()
    ctx = dbie.DBIE(wl.nx, wl.ny, wl.h, wl.x0, wl.y0, *hb, fp32=True); ctx.eval_f32_host(hxn, hyn, hzn, hln); ctx.close()
    t0 = time.perf_counter()
    for k in range(steps):
        ctx = dbie.DBIE(wl.nx, wl.ny, wl.h, wl.x0, wl.y0, *hb, fp32=True)
        o = ctx.eval_f32_host(hxn, hyn, hzn, hln)
        ctx.close()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    try:
        dfma_meas, ffma_meas = dbie.probe_dfma_rate(300.0)
    except Exception:
        dfma_meas = ffma_meas = None
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak = SM_COUNT * MUFU_LANES_PER_SM * sm_max * 1e6
    kern_ips = inter * steps / (kern_ms * 1e-3) if kern_ms > 0 else 0.0
    ach = kern_ips * MUFU_PER_INTERACTION
    return {
        "metric": "point-pixel DBIE interactions/sec (fp32)", "value": inter * steps / (ms_total * 1e-3),
        "unit": UNIT, "n_gpus": 1, "steps": steps, "warmup": warmup, "ms_per_step": ms_total / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": dict(workload_config(wl, Mode("cfg4")), step="dbie_create(DBIE_WITH_FP32) + dbie_eval_f32"),
        "clocks": clocks,
        "e2e": {"value": inter * steps / (e2e_ms * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": 3 * wl.N * 8 + 6 * wl.M * 4, "d2h_bytes_per_step": 3 * wl.M * 4,
                "ms_per_step": e2e_ms / steps, "api": "dbie_create_host(DBIE_WITH_FP32) + dbie_eval_f32_host"},
        "gpu_launches": launches,
        "roofline": {"bound": "alu", "kernel": "dbie::interact_f32_kernel",
                     "kernel_what": "fp32 point-pixel sums, SFU sincos of the reduced argument",
                     "achieved": 1e-12 * ach, "peak": 1e-12 * peak, "unit": "T MUFU lane-op/s", "frac": ach / peak,
                     "traffic": (ncu_traffic().get("f32") or {}).get("dram_bytes_per_launch") if points == 0 else None,
                     "traffic_source": (ncu_traffic().get("f32") or {}).get("capture"),
                     "mufu_per_interaction": MUFU_PER_INTERACTION,
                     "note": "SFU-bound: 148 SM x 16 MUFU lanes x clocks.max.sm / 7 MUFU per interaction (the issue port, 40 "
                             "instructions per interaction, allows 40 % more; the FP32 FMA pipe 75 % more; profiles/r02_sass_loops.txt)",
                     "kernel_interactions_per_s": kern_ips, "kernel_ms_per_launch": kern_ms / max(kern_launches, 1),
                     "kernel_launches": kern_launches, "kernel_share_of_step": kern_ms / ms_total if ms_total else None,
                     "peak_measured_ffma_per_s": ffma_meas},
        "cpu_baseline": None,
    }


def measure_slabs(steps: int) -> dict:
    """the full 256x256x128 volume is hours even at the roofline, so time z-slabs of
    256 x 256 = 65,536 points at a few heights and project.  GRID, T = 8, 10 levels, Eq. 13 differences."""
    import torch
    import workloads
    import paper_1306_1122_b200 as dbie
    dev = torch.device("cuda", 0)
    full = workloads.config5()
    nlay = 128
    per = full.M // nlay
    assert per == 65536
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(dev)
    ctx = dbie.DBIE(full.nx, full.ny, full.h, full.x0, full.y0, t(full.bx), t(full.by), t(full.bz))
    ctx.profile(True)
    sopts = dbie.default_opts(method=1)
    out = []
    sampler = ClockSampler(0)
    for layer in (0, 31, 127):                      # z = 1, 32, 128 pixels
        idx = np.arange(layer * per, (layer + 1) * per)
        sub = full.subset(idx)
        dx, dy, dz = t(sub.x), t(sub.y), t(sub.z)
        best = None
        for k in range(max(steps, 1)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            s = ctx.solve(dx, dy, dz, sopts)
            e1.record(); e1.synchronize()
            ms = e0.elapsed_time(e1)
            c = ctx.counters(); kt = ctx.kernel_time()
            rec = {"z_px": float(sub.z[0] / full.h), "points": per, "ms": ms, "interactions": c["interactions"],
                   "value": c["interactions"] / (ms * 1e-3), "kernel_ms": kt["interact_ms"],
                   "levels_mean": float(s["iters"].double().mean().item()),
                   "status0_frac": float((s["status"] == 0).double().mean().item()),
                   "mean_f": float(s["f"].mean().item()), "mean_g": float(s["g"].mean().item())}
            if best is None or rec["ms"] < best["ms"]:
                best = rec
        out.append(best)
    ctx.close()
    clocks = sampler.stop()
    peak = SM_COUNT * FP64_LANES_PER_SM * ((clocks or {}).get("sm_max_mhz") or 1965.0) * 1e6   # the sampled clocks.max.sm
    for rec in out:
        rec["roofline_frac_kernel"] = rec["interactions"] / (rec["kernel_ms"] * 1e-3) * FP64_INSTR["grid"] / peak
    mean_ms = float(np.mean([r["ms"] for r in out]))
    return {"clocks": clocks, "workload": "BASELINE configs[4] z-slabs: 256x256 points at z = 1, 32, 128 px, 1024x1024 boundary, GRID T=8, 10 levels",
            "slabs": out, "projected_full_volume_s": mean_ms * 1e-3 * nlay,
            "note": "full volume (128 slabs, 8,388,608 points) NOT run: projected = mean slab time x 128"}


def run_ours(args, mode: Mode) -> None:
    import torch
    import paper_1306_1122_b200 as dbie
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        # the communicator lines (rank / nranks) of NCCL's start-up let a reader of the log check the world size
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local)
    dbie.load()

    detail = args.detail or ("gpurun_out/bench_detail.json" if args.legs else "")
    if args.dtype == "f32":
        if rank == 0:
            emit(measure_f32(args.steps, args.warmup, args.points), detail)
        return
    if args.slabs:
        if rank == 0:
            print(json.dumps(_sig(measure_slabs(args.steps))), flush=True)
        return

    line = measure_f64(mode, args.steps, args.warmup, rank, world, local, dist)
    if rank == 0:
        base = (cpu_baseline(make_workload(mode.workload, points=mode.points), mode, target_s=args.cpu_seconds)
                if args.cpu_seconds > 0 else None)
        line["cpu_baseline"] = base
        if base:
            line["gpu_over_cpu_baseline"] = line["value"] / base["value"]
        headline_default = mode.workload == "cfg4" and mode.points == 0 and not mode.analytic
        if headline_default:
            line["vs_previous_round"] = {"cfg4_eval": line["value"] / PREVIOUS_ROUND["cfg4_eval"]}
        if world == 1 and headline_default and args.also:
            # BASELINE configs[1] in the same run (two steps): the Nelder-Mead solve stays comparable round over round
            ls, lw = max(1, min(args.steps, 2)), max(1, min(args.warmup, 3))
            legs = {"cfg2_nm": measure_f64(Mode("cfg2"), ls, lw, e2e=False)}
            if args.legs:
                # small-batch latency (what a line tracer calls): 48 points, the warp-per-point shape of the fused kernel
                legs["cfg2_nm_48pts"] = measure_f64(Mode("cfg2", points=48), 5, 3)
                legs["cfg5_grid"] = measure_f64(Mode("cfg5", grid=True, points=8192), 1, 1)
                legs["cfg4_f32"] = measure_f32(ls, lw)
                legs["cfg4_f64_reduced_sincos"] = measure_f64(Mode("cfg4", reduced=True), ls, lw)
            line["legs"] = legs
            line["also"] = {k: {"value": v["value"], "ms_per_step": v["ms_per_step"], "frac": v["roofline"]["frac"]}
                            for k, v in legs.items()}
            line["vs_previous_round"]["cfg2_nm"] = legs["cfg2_nm"]["value"] / PREVIOUS_ROUND["cfg2_nm"]
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
        if rank == 0:
            time.sleep(1.0)      # NCCL's INFO lines of the other ranks' teardown come first: the headline stays the LAST line
    if rank == 0:
        emit(line, detail)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=["cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--method", default=None, choices=["nm", "grid"],
                    help="lambda search of the solve workloads (default: nm; cfg5: grid)")
    ap.add_argument("--gradient", default="fd", choices=["fd", "analytic"],
                    help="solve workloads: Eq. 13 finite differences (the paper's) or the analytic gradient (O-5)")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"],
                    help="f32: the dbie_eval_f32 leg of BASELINE configs[3] alone (implies --workload cfg4, one GPU)")
    ap.add_argument("--points", type=int, default=0,
                    help="solve/eval a seeded subset of this many points (0: the whole volume; cfg5: 16384)")
    ap.add_argument("--slabs", action="store_true",
                    help="config 5 as SURVEY 8(d) asks: GRID solve of three 65,536-point z-slabs + projected full-volume time")
    ap.add_argument("--legs", action="store_true",
                    help="default workload on one GPU: also time the 48-point latency, config-5 GRID, fp32 and reduced-sincos "
                         "legs; their full records go to the --detail file, their values into the line's `also`")
    ap.add_argument("--no-also", dest="also", action="store_false",
                    help="default workload: skip the two-step config-2 Nelder-Mead leg reported under `also`")
    ap.add_argument("--detail", default="",
                    help="also write the full record (every diagnostic field) to this file")
    ap.add_argument("--cpu-seconds", type=float, default=15.0,
                    help="target CPU time of the cpu_baseline leg (0 disables it)")
    args = ap.parse_args()
    if args.workload != "cfg4":
        args.legs = False
        args.also = False
    mode = Mode(args.workload, grid=(args.method == "grid") or (args.method is None and args.workload == "cfg5"),
                analytic=args.gradient == "analytic", points=args.points)
    if args.impl == "reference":
        run_reference(args, mode)
    else:
        if args.gpus > 1 and int(os.environ.get("WORLD_SIZE", "1")) == 1:
            # convenience: re-launch under torchrun, one rank per GPU
            cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
                   "--master-addr", "127.0.0.1", "--master-port", "29541", os.path.abspath(__file__)] + sys.argv[1:]
            raise SystemExit(subprocess.call(cmd))
        run_ours(args, mode)


if __name__ == "__main__":
    main()
