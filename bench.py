#!/usr/bin/env python
"""bench.py — headline measurement of hard-b200 (contract: see the task statement / DESIGN.md §Measurement).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl cuda|reference]
                  [--workload c4|c3|c2s] [--scheme A|B] [--variant fused|perdir]
                  [--no-e2e] [--no-cpu-baseline] [--no-variants] [--no-ncu-traffic]

One "step" = one Heun / SSP-RK2 step of the whole hot path (ghost fill, stage 1, ghost fill, stage 2
with the fused CFL reduction) over the workload's full mesh.  Metric (BASELINE.json): fp64 cell-updates
per second per RK stage = cells * 2 * K / time.  Default workload: C4 (BASELINE.json configs[4], 896^3
periodic seeded sine-mode field, CFL 0.4), scheme A (the paper's WENO5-Z + HLL + Heun).
N > 1: the path does not shard without a halo exchange that north_star excludes ("everything runs on
one GPU"), so N ranks run N independent replicas (replicas only), weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 cell-updates/sec per RK stage"
UNIT = "cell-stage-updates/s"
ALG_BYTES_PER_CELL_STAGE = 100.0     # stage 1 = 40 R + 40 W, stage 2 = 80 R + 40 W  => 100 B average
# roofline.frac (round 3) follows COUNTERS, not a chosen unit of work: the fp64-pipe instructions the stage kernel
# actually EXECUTED per launch (ncu sm__inst_executed_pipe_fp64.sum x 32 lanes, collected by the ncu child run of
# this same bench; a count, never a time) x 2 flop / the live CUDA-event launch time / the live DFMA peak.
# Units of work one can divide by instead, all per cell-stage, fp64-pipe thread instructions:
#   935   scheme A, what the committed device functions need with no redundancy (halo items, idle lanes)
#   1 104 / 1 152   scheme A, executed by stage 1 / stage 2 (ncu, round-2 kernels; the fallback below)
#   1 300 round 1's hand count, the unit `frac` used in rounds 1-2 -> now reported as work_unit_frac only
#   1 700 - 1 900   SURVEY.md section 8(d)'s estimate (+-30 %; too high: it would put the kernel above the peak)
WORK_UNIT_FP64_PER_CELL_STAGE = {"A": 1300.0, "B": 540.0}
MINIMAL_FP64_PER_CELL_STAGE = {"A": 935.0, "B": None}
# executed counts of the committed kernels from profiles/ (average of the two stage launches), used only when ncu
# cannot run inside bench.py (missing binary, closed counters); the line then says so in roofline.frac_source
FALLBACK_EXECUTED_FP64 = {"A": 1128.0, "B": 404.0}

WORKLOADS = {"c4": (896, 10), "c3": (512, 20), "c2s": (256, 10)}
# BASELINE.json configs[0..2]: launch-bound meshes ("run to t" configs; timed here over a fixed number of steps from
# the initial state, CUDA-graph replay on, as Hard.run_to drives them).  name -> (generator, steps per --steps unit)
LAUNCH_BOUND = {"c0": ("sod", 1000, 200), "c1": ("leblanc", 4096, 200), "c2": ("sedov", 128, 2)}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="c4", choices=sorted(WORKLOADS) + sorted(LAUNCH_BOUND))
    ap.add_argument("--scheme", default="A", choices=["A", "B"])
    ap.add_argument("--variant", default="fused", choices=["fused", "perdir"])
    ap.add_argument("--radiation", action="store_true", help="NEXT-1: carry E_rad as a sixth advected field")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: split ONE mesh into z-slabs with halo exchange (NEXT-4, strong scaling) instead of replicas")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-variants", action="store_true",
                    help="skip the short extra measurements of the per-direction variant and of the other scheme")
    ap.add_argument("--no-ncu-traffic", action="store_true",
                    help="do not measure roofline.traffic (DRAM bytes of the stage kernel) with an ncu child run")
    return ap.parse_args()


# ------------------------------------------------------------------------------------ ranks
def max_over_ranks(x, device="cpu"):
    """Max of a python float over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(cells_per_rank, stages, steps, ms_max, world):
    """Whole-job cell-stage-updates/s of `world` replicas that each did cells*stages*steps in ms_max."""
    return world * cells_per_rank * float(stages) * steps / (ms_max * 1e-3)


# ------------------------------------------------------------------------------------ clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, pw, mx, reasons = [], [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for (t, line) in self.rows:
            if t < t0 or t > t1 + 0.1:
                continue
            p = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(p[0]))
                mx = float(p[1])
            except Exception:
                continue
            try:
                pw.append(float(p[2]))
            except Exception:
                pass
            for nm, v in zip(names, p[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        pw.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm), "power_w": pw[len(pw) // 2] if pw else None}


# ------------------------------------------------------------------------------------ oracle legs
def oracle_rate(scheme, n, steps, warmup=0):
    """Times the oracle AS IT STANDS (single-threaded C++) on the same seeded sine-mode recipe at n^3."""
    import oracle
    from paper_2509_08971_b200 import workloads as wl
    w = wl.turbulence(n, nsteps=steps)
    o = oracle.Oracle(*w.n, w.gamma, w.bc, scheme=0 if scheme == "A" else 1, spacing=w.spacing)
    o.set_state(*w.state)
    if warmup:
        o.step(w.cfl, warmup)
    t0 = time.perf_counter()
    o.step(w.cfl, steps)
    dt = time.perf_counter() - t0
    o.close()
    return n ** 3 * 2 * steps / dt, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = 96
    value, secs = oracle_rate(args.scheme, n, args.steps, args.warmup)
    sample = ("oracle/hard_oracle.cpp, 1 thread, %d^3 periodic box of the same seeded sine-mode recipe "
              "(a bounded sample: the full %s mesh needs hours), %d+%d steps" % (n, args.workload, args.warmup, args.steps))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "%s scheme %s (oracle sample %d^3)" % (args.workload, args.scheme, n)},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ DRAM traffic (ncu child run)
NCU_METRICS = ("dram__bytes_read.sum", "dram__bytes_write.sum", "sm__inst_executed_pipe_fp64.sum",
               "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "smsp__inst_executed.sum",
               "smsp__issue_active.avg.pct_of_peak_sustained_active")


def ncu_stage_counters(args, timeout=300):
    """Counters of the stage kernel per launch, measured by running this same bench (2 steps, nothing else) as a
    child under ncu and averaging the stage-1 and stage-2 launches of the second step: DRAM bytes (roofline.traffic),
    executed fp64-pipe and total warp instructions, fp64-pipe and issue utilisation.  Only counters come from the
    profiled run — never a time.  (None, why) if ncu is missing, closed on the pool, or the child fails."""
    import shutil
    import signal
    import tempfile
    ncu = shutil.which("ncu") or "/usr/local/cuda/bin/ncu"
    if not os.path.exists(ncu):
        return None, "ncu not found"
    log = tempfile.NamedTemporaryFile(prefix="hard_ncu_", suffix=".csv", delete=False).name
    cmd = [ncu, "--metrics", ",".join(NCU_METRICS), "--clock-control", "none", "--print-units", "base",
           "-k", "regex:stage", "-s", "2", "-c", "2", "--csv", "--log-file", log,
           sys.executable, os.path.abspath(__file__), "--workload", args.workload, "--scheme", args.scheme,
           "--variant", "fused", "--steps", "2", "--warmup", "0", "--no-e2e", "--no-cpu-baseline", "--no-variants",
           "--no-ncu-traffic"] + (["--radiation"] if args.radiation else [])
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK=os.environ.get("LOCAL_RANK", "0"))
    try:
        p = subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, env=env, start_new_session=True)
        try:
            out, _ = p.communicate(timeout=timeout)
        except subprocess.TimeoutExpired:
            os.killpg(p.pid, signal.SIGKILL)
            return None, "ncu child run timed out"
        if p.returncode != 0:
            return None, "ncu child run failed: " + (out or "").strip().splitlines()[-1][:160] if out else "ncu child run failed"
        import csv
        rows = [r for r in csv.reader(open(log)) if len(r) > 6]
        H = rows[0]
        per_launch = {}
        for r in rows[1:]:
            d = dict(zip(H, r))
            per_launch.setdefault(d["ID"], {})[d["Metric Name"]] = float(d["Metric Value"].replace(",", ""))
        if len(per_launch) != 2 or any(set(NCU_METRICS) - set(m) for m in per_launch.values()):
            return None, "ncu child run captured %d stage launches (expected 2) or lacks a metric" % len(per_launch)
        avg = {k: sum(m[k] for m in per_launch.values()) / 2.0 for k in NCU_METRICS}
        out = {"traffic": avg["dram__bytes_read.sum"] + avg["dram__bytes_write.sum"],
               "fp64_warp_inst": avg["sm__inst_executed_pipe_fp64.sum"],
               "fp64_pipe_busy_pct": avg["sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"],
               "warp_inst": avg["smsp__inst_executed.sum"],
               "issue_active_pct": avg["smsp__issue_active.avg.pct_of_peak_sustained_active"]}
        return out, "measured in this run: " + " ".join(cmd[:2]) + " <6 counters> " + " ".join(cmd[3:13]) + " ... (child bench, 2 steps)"
    except Exception as ex:
        return None, "ncu child run: %s" % str(ex)[:160]
    finally:
        try:
            os.unlink(log)
        except OSError:
            pass


# ------------------------------------------------------------------------------------ launch-bound configs
def launch_bound_measure(name, scheme, units, warm_units, local):
    """C0 / C1 / C2 (BASELINE.json configs[0..2]): K = units * steps-per-unit Heun steps from the initial state on
    torch's current (capturable) stream, so hard_step replays its two-step CUDA graph; device-timed with CUDA events.
    The state is tiny (C0: 40 KB) and lives in L2: the figure is launch latency, not bandwidth — reported as such."""
    import torch
    from paper_2509_08971_b200 import hard
    from paper_2509_08971_b200 import workloads as wl
    gen, n, per = LAUNCH_BOUND[name]
    w = getattr(wl, gen)(n)
    k = max(units, 1) * per
    h = hard.Hard(*w.n, w.gamma, w.bc, scheme=hard.SCHEME_WENO5Z_HLL if scheme == "A" else hard.SCHEME_MUSCL_HLLC, spacing=w.spacing)
    st = [torch.from_numpy(__import__("numpy").ascontiguousarray(a)).cuda() for a in w.state]
    h.set_state(*st)
    h.step(w.cfl, max(warm_units, 1) * per)              # warm-up: graph capture + instantiation happen here
    h.set_state(*st)
    stream = torch.cuda.current_stream()
    smp = ClockSampler(local)
    smp.start()
    time.sleep(0.3)
    l0 = h.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t0 = time.time()
    e0.record(stream)
    h.step(w.cfl, k)
    e1.record(stream)
    torch.cuda.synchronize()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    t_sim, steps_done = h.time()                         # surfaces a latched non-physical state
    cells = w.n[0] * w.n[1] * w.n[2]
    out = {"value": cells * 2.0 * k / (ms * 1e-3), "unit": UNIT, "workload": "%s %s" % (name, w.name), "cells": cells,
           "steps": k, "us_per_step": ms * 1e3 / k, "ms_per_step": ms / k, "gpu_launches": h.launch_count() - l0,
           "graph_replay": os.environ.get("HARD_NO_GRAPH") is None, "sim_time": t_sim, "steps_done": steps_done,
           "clocks": smp.stop(t0, t1)}
    h.close()
    return out


def run_launch_bound(args):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:                                      # a 1 000-cell mesh does not shard: rank 0 alone measures it
        return
    if not torch.cuda.is_available():
        print("bench.py: no CUDA device; the CUDA path has no CPU fallback", file=sys.stderr, flush=True)
        raise SystemExit(3)
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    m = launch_bound_measure(args.workload, args.scheme, args.steps, args.warmup, local)
    line = {"metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": 1, "steps": m["steps"], "warmup": args.warmup * LAUNCH_BOUND[args.workload][2],
            "ms_per_step": m["ms_per_step"], "us_per_step": m["us_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": m["workload"] + " (BASELINE.json configs[%s]); launch-bound: 4 launches per step, CUDA-graph replay of two steps" % args.workload[1],
                       "scheme": args.scheme, "l2": "state fits in L2 by design of the config; the figure is launch latency"},
            "roofline": None, "roofline_note": "launch-latency bound (DESIGN.md section 1): no bandwidth or ALU roofline applies",
            "e2e": None, "cpu_baseline": None, "clocks": m["clocks"], "gpu_launches": m["gpu_launches"]}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2509_08971_b200 import hard
    from paper_2509_08971_b200 import workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    has_cuda = torch.cuda.is_available()
    if has_cuda:
        torch.cuda.set_device(local)
    if world > 1:                                  # the communicator comes up first (gloo on a box without GPUs)
        if has_cuda:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
    if not has_cuda:
        msg = "bench.py: no CUDA device; the CUDA path has no CPU fallback"
        if world > 1:
            from paper_2509_08971_b200 import sharded
            comm = sharded.DistComm(True)          # the z-slab neighbour map and pairing code of --shard
            dist.barrier()
            msg += " (communicator up: world %d, backend %s, rank %d, z-slab neighbours %s, slab %s of nz=%d)" % (
                comm.world, dist.get_backend(), comm.rank, (comm.lo, comm.hi),
                sharded.split_z(WORKLOADS[args.workload][0], world)[rank], WORKLOADS[args.workload][0])
            dist.destroy_process_group()
        print(msg, file=sys.stderr, flush=True)
        raise SystemExit(3)
    dev = torch.device("cuda", local)

    n, _cfg_steps = WORKLOADS[args.workload]
    K, W = args.steps, args.warmup
    scheme = hard.SCHEME_WENO5Z_HLL if args.scheme == "A" else hard.SCHEME_MUSCL_HLLC
    variant = hard.VARIANT_FUSED if args.variant == "fused" else hard.VARIANT_PERDIR
    w = wl.turbulence(n, nsteps=K, device=dev)
    cells = n ** 3
    shard = args.shard and world > 1 and not args.radiation and variant == hard.VARIANT_FUSED
    if shard:
        from paper_2509_08971_b200 import sharded
        sh = sharded.ShardedHard(w.n, w.gamma, w.bc, scheme=scheme, spacing=w.spacing)
        h = sh.slab.h
        slab_cells = n * n * (sh.slab.k1 - sh.slab.k0)
        set_state = lambda: sh.set_state(w.state)
        do_step = lambda k: sh.step(w.cfl, k)
    else:
        h = hard.Hard(*w.n, w.gamma, w.bc, scheme=scheme, variant=variant, spacing=w.spacing, radiation=args.radiation)
        slab_cells = cells
        set_state = lambda: h.set_state(*w.state)
        do_step = lambda k: h.step(w.cfl, k)
    stream = torch.cuda.current_stream()
    nfields = 6 if args.radiation else 5
    alg_bytes = ALG_BYTES_PER_CELL_STAGE * nfields / 5.0
    e_rad = (1.0 + 0.3 * w.state[0]) if args.radiation else None      # seeded, positive, non-uniform

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: inputs already in HBM when the timed region starts
    set_state()
    if args.radiation:
        h.set_rad_energy(e_rad)
    do_step(W)                             # warm-up steps (untimed)
    set_state()                            # timed steps are exactly the workload's steps 1..K
    if args.radiation:
        h.set_rad_energy(e_rad)
    fp64_peak = hard.probe_fp64_peak()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    launches0 = h.launch_count()
    h.stage_time(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.time()
    e0.record(stream)
    do_step(K)
    e1.record(stream)
    barrier()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    stage_ms, stage_launches = h.stage_time(reset=False)
    launches = h.launch_count() - launches0
    clocks = sampler.stop(t0, t1)
    t_sim, steps_done = h.time()
    ms = max_over_ranks(ms, dev)
    value = job_throughput(cells, 2, K, ms, 1 if shard else world)

    # ---- roofline of the dominant kernel (the stage kernel), live CUDA-event durations
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    per_launch_ms = stage_ms / max(stage_launches, 1)
    if variant == hard.VARIANT_FUSED:
        cell_stages_per_launch = slab_cells                  # one launch = one RK stage over the (local) mesh
    else:
        cell_stages_per_launch = cells * 2.0 * K / max(stage_launches, 1)
    alg_gbs = cell_stages_per_launch * alg_bytes / (per_launch_ms * 1e-3) / 1e9
    def tflops(fp64_per_cell_stage):
        return cell_stages_per_launch * 2.0 * fp64_per_cell_stage / (per_launch_ms * 1e-3) / 1e12

    executed = FALLBACK_EXECUTED_FP64[args.scheme] * (6.0 / 5.0 if args.radiation else 1.0)
    work_unit = WORK_UNIT_FP64_PER_CELL_STAGE[args.scheme] * (6.0 / 5.0 if args.radiation else 1.0)
    unit_tflops = tflops(work_unit)
    roofline = {"bound": "alu", "kernel": ("stage3d_kernel<%s, %d, stage 1|2>" % (args.scheme, nfields)) if variant == hard.VARIANT_FUSED else ("stage_kernel<%s, %d> per direction + axpy_kernel" % (args.scheme, nfields)),
                "achieved": tflops(executed), "peak": fp64_peak,
                "unit": "TFLOP/s", "frac": tflops(executed) / fp64_peak if fp64_peak else None,
                "frac_source": "executed fp64-pipe instructions per cell-stage from profiles/ (ncu did not run inside this bench)",
                "executed_fp64_per_cell_stage": executed, "fp64_pipe_busy_pct": None, "issue_active_pct": None,
                "warp_inst_per_cell_stage": None,
                "work_unit_frac": unit_tflops / fp64_peak if fp64_peak else None,
                "work_unit_fp64_per_cell_stage": work_unit,
                "minimal_fp64_per_cell_stage": MINIMAL_FP64_PER_CELL_STAGE[args.scheme],
                "useful_frac": (tflops(MINIMAL_FP64_PER_CELL_STAGE[args.scheme]) / fp64_peak)
                               if (fp64_peak and MINIMAL_FP64_PER_CELL_STAGE[args.scheme] and not args.radiation) else None,
                "units_note": "per cell-stage, fp64-pipe thread instructions (1 instruction = 2 flop, the DFMA peak's unit): "
                              "frac uses what the kernel executed (ncu); work_unit_frac the fixed round-1 hand count "
                              "(SURVEY 8(d) estimated 1700-1900 for A, too high); useful_frac the count with no redundancy",
                "traffic": None, "traffic_note": "not measured in this run",
                "alg_bytes_per_launch": slab_cells * alg_bytes,
                "peak_source": "measured live: hard_probe_fp64_peak (DFMA chains on all SMs, libhard_probe.so)",
                "avg_launch_ms": per_launch_ms, "launches_timed": stage_launches}
    roofline_hbm = {"bound": "hbm", "achieved": alg_gbs, "peak": hbm_peak, "unit": "GB/s", "frac": alg_gbs / hbm_peak,
                    "frac_of_nominal_8TBs": alg_gbs / 8000.0, "peak_source": hbm_src,
                    "alg_bytes_per_cell_stage": alg_bytes}

    # ---- end to end through the C-ABI with HOST buffers (pinned): H2D + K steps + D2H inside the timed region
    e2e = None
    if not args.no_e2e and not args.radiation and not shard:
        try:
            import psutil
            need = 2 * 5 * cells * 8                       # pinned input + output copies of the state
            avail = psutil.virtual_memory().available / max(world, 1)
            if avail < 1.3 * need:
                raise MemoryError("host memory: %.0f GB available per rank, %.0f GB of pinned buffers needed"
                                  % (avail / 1e9, need / 1e9))
            host_in = [torch.empty((n, n, n), dtype=torch.float64, pin_memory=True) for _ in range(5)]
            for a, b in zip(host_in, w.state):
                a.copy_(b)
            host_out = [torch.empty((n, n, n), dtype=torch.float64, pin_memory=True) for _ in range(5)]
            w.state = None
            torch.cuda.empty_cache()
            barrier()
            te0 = time.perf_counter()
            h.set_state(*host_in)           # host -> device (5 pitched copies) + CFL pass
            h.step(w.cfl, K)
            h.get_state(host_out)           # device -> host, synchronises
            torch.cuda.synchronize()
            te = time.perf_counter() - te0
            te = max_over_ranks(te, dev)
            nbytes = 5 * cells * 8
            e2e = {"value": job_throughput(cells, 2, K, te * 1e3, world), "unit": UNIT, "h2d_bytes_per_step": nbytes / K,
                   "d2h_bytes_per_step": nbytes / K, "seconds": te,
                   "what": "hard_set_state(host pinned) + hard_step(cfl, %d) + hard_get_state(host pinned); "
                           "the state crosses PCIe once per %d-step job" % (K, K)}
            del host_in, host_out
        except Exception as ex:                      # e.g. not enough pinned host memory on the box
            e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0, "error": str(ex)[:200]}
    h.close()
    del h
    w.state = None
    torch.cuda.empty_cache()

    # ---- short side measurements in the same run (BASELINE.json configs[4]: "fused vs per-direction kernels"):
    # the per-direction variant of this scheme and the fused kernel of the other scheme, device-resident, CUDA events
    variants = None
    if rank == 0 and world == 1 and not args.no_variants and not args.radiation and variant == hard.VARIANT_FUSED:
        variants = {}
        other = "B" if args.scheme == "A" else "A"
        n3, _ = WORKLOADS["c3"]
        # name, mesh, scheme, variant, steps, sixth field: every number BASELINE.md section 4 quotes has a twin here,
        # each with its own clock record (sampled over its own timed region)
        for name, nn, sch, var, k, rad in (("perdir_" + args.scheme, n, args.scheme, hard.VARIANT_PERDIR, 3, False),
                                           ("fused_" + other, n, other, hard.VARIANT_FUSED, max(3, K // 2), False),
                                           ("perdir_" + other, n, other, hard.VARIANT_PERDIR, 3, False),
                                           ("fused_A6_c3", n3, "A", hard.VARIANT_FUSED, 5, True)):
            try:
                wv = wl.turbulence(nn, nsteps=k, device=dev)
                hv = hard.Hard(*wv.n, wv.gamma, wv.bc, scheme=hard.SCHEME_WENO5Z_HLL if sch == "A" else hard.SCHEME_MUSCL_HLLC,
                               variant=var, spacing=wv.spacing, radiation=rad)
                er = (1.0 + 0.3 * wv.state[0]) if rad else None

                def load():
                    hv.set_state(*wv.state)
                    if rad:
                        hv.set_rad_energy(er)
                load()
                hv.step(wv.cfl, 1)
                load()
                l0 = hv.launch_count()
                smp = ClockSampler(local)
                smp.start()
                time.sleep(0.3)
                ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                tv0 = time.time()
                ev0.record(stream)
                hv.step(wv.cfl, k)
                ev1.record(stream)
                torch.cuda.synchronize()
                tv1 = time.time()
                msv = ev0.elapsed_time(ev1)
                hv.time()                                  # surfaces a latched non-physical state
                nc = nn ** 3
                variants[name] = {"value": nc * 2.0 * k / (msv * 1e-3), "unit": UNIT, "steps": k, "warmup": 1,
                                  "workload": "%d^3" % nn, "fields": 6 if rad else 5,
                                  "ms_per_step": msv / k, "gpu_launches": hv.launch_count() - l0,
                                  "alg_GBs": nc * (240.0 if rad else 200.0) * k / (msv * 1e-3) / 1e9,
                                  "clocks": smp.stop(tv0, tv1)}
                hv.close()
                del hv, wv, er
                torch.cuda.empty_cache()
            except Exception as ex:
                variants[name] = {"value": None, "error": str(ex)[:200]}
        # NEXT-4 on the one GPU there is: the same mesh as two z-slabs of 448 planes emulated in this process
        # (sharded.LocalGroup: the ranks' phases in lockstep, halos packed, copied device-to-device and unpacked, lambda
        # max-reduced in place, exactly the sequence ShardedHard.step runs over NCCL).  Not a scaling number: it shows
        # what the pack / unpack / reduction and the split stage launches cost per step next to the single domain.
        try:
            from paper_2509_08971_b200 import sharded
            k = 3
            wv = wl.turbulence(n, nsteps=k, device=dev)
            grp = sharded.LocalGroup(wv.n, wv.gamma, wv.bc, 2, scheme=scheme, spacing=wv.spacing)
            grp.set_state(wv.state)
            grp.step(wv.cfl, 1)
            grp.set_state(wv.state)
            l0 = sum(sl.h.launch_count() for sl in grp.slabs)
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            ev0.record(stream)
            grp.step(wv.cfl, k)
            ev1.record(stream)
            torch.cuda.synchronize()
            msv = ev0.elapsed_time(ev1)
            for sl in grp.slabs:
                sl.h.time()
            variants["sharded_local_2x%d_%s" % (n // 2, args.scheme)] = {
                "value": cells * 2.0 * k / (msv * 1e-3), "unit": UNIT, "steps": k, "warmup": 1, "workload": "%d^3 as 2 z-slabs on ONE GPU" % n,
                "ms_per_step": msv / k, "overhead_ms_per_step_vs_single_domain": msv / k - ms / K,
                "gpu_launches": sum(sl.h.launch_count() for sl in grp.slabs) - l0,
                "halo_bytes_per_step": 2 * 2 * 2 * grp.slabs[0].h.halo_doubles() * 8,
                "note": "LocalGroup emulation (no NCCL, one process); not a multi-GPU measurement"}
            for sl in grp.slabs:
                sl.close()
            del grp, wv
            torch.cuda.empty_cache()
        except Exception as ex:
            variants["sharded_local_2"] = {"value": None, "error": str(ex)[:200]}
        for lb in ("c0", "c1", "c2"):                      # BASELINE.json configs[0..2]: launch-bound, us per step
            try:
                variants[lb + "_" + args.scheme] = launch_bound_measure(lb, args.scheme, 5, 1, local)
            except Exception as ex:
                variants[lb + "_" + args.scheme] = {"value": None, "error": str(ex)[:200]}

    if rank == 0 and world == 1 and not args.no_ncu_traffic and variant == hard.VARIANT_FUSED and not shard:
        ctr, note = ncu_stage_counters(args)
        roofline["traffic_note"] = note + "; average of one stage-1 and one stage-2 launch; algorithmic bytes per launch in alg_bytes_per_launch"
        if ctr is not None:
            roofline["traffic"] = ctr["traffic"]
            executed = ctr["fp64_warp_inst"] * 32.0 / cells
            roofline.update({"achieved": tflops(executed), "frac": tflops(executed) / fp64_peak if fp64_peak else None,
                             "frac_source": "executed fp64-pipe instructions of this run's ncu child (sm__inst_executed_pipe_fp64.sum x 32 "
                                            "lanes per launch) x 2 flop / live CUDA-event launch time / live DFMA peak",
                             "executed_fp64_per_cell_stage": executed, "fp64_pipe_busy_pct": ctr["fp64_pipe_busy_pct"],
                             "issue_active_pct": ctr["issue_active_pct"], "warp_inst_per_cell_stage": ctr["warp_inst"] * 32.0 / cells})

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        nb, sb = 128, 3
        v, secs = oracle_rate(args.scheme, nb, sb)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": secs,
                        "sample": "oracle/hard_oracle.cpp as it stands, 1 thread, %d Heun steps of the same seeded "
                                  "sine-mode recipe at %d^3 (the %d^3 mesh would take hours)" % (sb, nb, n)}
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": "%s: %d^3 periodic seeded sine-mode field, CFL %.2g, %d Heun steps" % (args.workload, n, w.cfl, K),
                           "scheme": "A: WENO5-Z + HLL + Heun (PAPER.md P:151)" if args.scheme == "A" else "B: MUSCL-minmod + HLLC + SSP-RK2 (north_star fallback)",
                           "variant": args.variant, "fields": nfields, "parallelism": ("z-slabs x%d (halo exchange + all-reduce max)" % world) if shard else ("replicas x%d" % world),
                           "l2": "state (%.1f GB per buffer) is far larger than the 126 MB L2; no flush needed" % (5 * cells * 8 / 1e9),
                           "sim_time": t_sim, "steps_done": steps_done},
                "roofline": roofline, "roofline_hbm": roofline_hbm, "e2e": e2e, "cpu_baseline": cpu_baseline,
                "variants": variants, "clocks": clocks, "gpu_launches": launches, "fp64_peak_tflops_measured": fp64_peak}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    elif args.workload in LAUNCH_BOUND:
        run_launch_bound(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
