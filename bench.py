"""bench.py -- throughput of the hyperbolic-relaxation hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config3] [--impl reference]

A "step" is one pass of the whole hot path (Alg. 1 l.9-16) over
the workload: the residual H + its L2 norm (a5) of the current state and one RK4 step = 4 x [fused RHS +
radiation condition + RK combine + inner ghost images (a1, a2, a4, a3), one launch]; the first
substep evaluates H anyway, so it also reduces the residual (hr_step_residual_async): 4 launches per step.  The one-time pieces (a0
source kernel, a6 step constants) run in hr_create, outside the timed region.

  metric  grid-point RK4 substep updates/s = N_int * 4 * K / (device time of K steps)
  value   fp64, state resident in HBM, timed with CUDA events on the solver's stream
  f32     the same workload in fp32 (BASELINE.json asks for both precisions)
  e2e     the same steps through the C ABI with HOST buffers: every step copies (u, v) from pinned
          host memory (hr_set_state, host pointers), runs the step and reads the residual back
  roofline  dominant kernel (the fused substep): algorithmic bytes 10 w per interior point-substep
           / mean launch duration measured here by hr_profile_step
  cpu_baseline  the CPU oracle (oracle/, test infrastructure) timed on this box's host cores

N > 1 (torchrun): the path does not shard ("replicas only"): every rank
advances an independent replica of the workload, no data-path collective; value = all ranks' units
/ max-over-ranks time.

`--impl reference` times the CPU oracle as it stands on the same workload, metric and unit (rank 0
only).  There is no installable reference for this paper.
"""
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

import numpy as np  # noqa: E402

import hr_workloads as W  # noqa: E402

METRIC = "grid-point RK4 substep updates/s"
UNIT = "point-substeps/s"


def workload(name: str) -> dict:
    if name.startswith("config"):
        return W.config(int(name[6:]))
    if name.startswith("sweep"):  # sweep<idx>:<N0>x<N1>x<N2>:<coord>:<order>
        idx, n, coord, order = name[5:].split(":")
        return W.sweep_point(int(idx), tuple(int(x) for x in n.split("x")), coord, int(order))
    raise SystemExit(f"unknown workload {name}")


def config_dict(p: dict, name: str, n_gpus: int) -> dict:
    ng = p["fd_order"] // 2
    T = [x + 2 * ng for x in p["n"]]
    ntot = T[0] * T[1] * T[2]
    return {"workload": f"BASELINE.json {name.replace('config', 'configs[') + ']' if name.startswith('config') else name}",
            "coord": p["coord"], "n_interior": list(p["n"]), "fd_order": p["fd_order"],
            "n_tot_points": ntot, "eta": p["eta"], "cfl": p["cfl"],
            "step": "residual (H + L2 norm) of the state + 1 RK4 step = 4 x (fused RHS+radiation+RK combine+ghost images, 1 launch each; the first also reduces the residual)",
            "l2": "inputs larger than L2 (10 grid functions = %.0f MB fp64)" % (10 * ntot * 8 / 1e6)
            if 10 * ntot * 4 > 126e6 else "working set fits L2 (%.1f MB fp64): L2 flushed between timed steps"
            % (10 * ntot * 8 / 1e6),
            "parallelism": "replicas only x%d" % n_gpus}


# ------------------------------------------------------------------------------------------------
# clocks during the timed region (profiling recipe's nvidia-smi line)
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 9:
                self.rows.append(f)

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for f in self.rows:
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
                power.append(float(f[3]))
            except ValueError:
                continue
            for nme, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm),
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# the CPU oracle legs (cpu_baseline and --impl reference): the only places that touch oracle/
# ------------------------------------------------------------------------------------------------
def oracle_step_seconds(p: dict, n_rk4: int, reps: int):
    """Seconds per [residual + n_rk4 RK4 steps] of the fp64 oracle on workload p, `reps` times."""
    from oracle import hr_oracle
    o = hr_oracle.Oracle(p)
    u = np.zeros(o.ntot)
    v = np.zeros(o.ntot)
    times = []
    for _ in range(reps):
        t0 = time.perf_counter()
        o.residual(u, 0)
        u, v = o.step(u, v, n_rk4)
        times.append(time.perf_counter() - t0)
    return times, o, hr_oracle.num_threads()


def cpu_baseline(p: dict, name: str) -> dict:
    t0 = time.perf_counter()
    times, o, threads = oracle_step_seconds(p, 1, 1)  # calibrate (also warms the pages)
    n = max(1, min(50, int(12.0 / max(times[0], 1e-3))))
    times, o, threads = oracle_step_seconds(p, 1, n)
    per = float(np.mean(times))
    out = {"value": o.n_int * 4 / per, "unit": UNIT, "cores": threads, "kind": "oracle",
           "sample": f"{n} x (residual + 1 RK4 step) of {name} in fp64 on the full grid, "
                     f"{per:.3f} s each, u = v = 0 start; total incl. oracle set-up "
                     f"{time.perf_counter() - t0:.1f} s"}
    # the single-thread figure SURVEY.md section 8(d) asks for beside the all-cores one: the same oracle in a child
    # process with OMP_NUM_THREADS=1, one warm-up + 2 timed (residual + RK4 step) on the same grid
    try:
        env = dict(os.environ, OMP_NUM_THREADS="1")
        r = subprocess.run([sys.executable, os.path.abspath(__file__), "--oracle-single", "--workload", name],
                           env=env, capture_output=True, text=True, timeout=600)
        single = json.loads(r.stdout.strip().splitlines()[-1])
        out["single_thread"] = {"value": single["value"], "unit": UNIT, "cores": single["cores"],
                                "sample": single["sample"]}
    except Exception as e:  # the all-cores figure stands on its own
        out["single_thread"] = {"unavailable": repr(e)[:200]}
    return out


def oracle_single(p: dict, name: str):
    times, o, threads = oracle_step_seconds(p, 1, 3)
    per = float(np.mean(times[1:]))
    print(json.dumps({"value": o.n_int * 4 / per, "cores": threads,
                      "sample": f"2 x (residual + 1 RK4 step) of {name}, fp64, full grid, {per:.3f} s each"}))


def run_reference(args, p, name):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import hr_oracle
    o = hr_oracle.Oracle(p)
    threads = hr_oracle.num_threads()
    u = np.zeros(o.ntot)
    v = np.zeros(o.ntot)

    def one():
        nonlocal u, v
        o.residual(u, 0)
        u, v = o.step(u, v, 1)

    for _ in range(args.warmup):
        one()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        one()
    dt = time.perf_counter() - t0
    value = o.n_int * 4 * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_dict(p, name, args.gpus),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                             "sample": f"{args.steps} x (residual + 1 RK4 step) of {name}, full grid, fp64"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# N > 1: replicas only.  No data-path collective: the only exchange is the
# maximum over ranks of the device time; value = all ranks' units / that time.
# ------------------------------------------------------------------------------------------------
def max_over_ranks(torch, sec: float, dist, device) -> float:
    if dist is None:
        return sec
    t = torch.tensor([sec], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replicas_value(world: int, n_int: int, steps: int, sec_max: float) -> float:
    """Whole-job point-substeps/s of `world` independent replicas that each did `steps` steps."""
    return world * n_int * 4 * steps / sec_max


# ------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------
MIN_TIMED_MS = 200.0  # the K-step block is repeated R times inside one event pair until the region is this long


def time_resident(torch, hr, p, dtype, steps, warmup, dist, flush_l2, min_ms=MIN_TIMED_MS):
    """K timed steps (x R repeats) with the state resident in HBM.
    Returns (seconds per K steps, max over ranks; solver; R)."""
    s = hr.Solver(p, dtype=dtype, residual_mode=0)
    out2 = torch.zeros(2, dtype=torch.float64, device=s.device)
    flush = None
    if flush_l2:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=s.device)

    def one():
        s.hr_step_residual_async(0, out2)  # residual of the state + one RK4 step (Alg. 1 l.9-16)

    def block(n):
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record(s.stream)
        for _ in range(n):
            one()
        e1.record(s.stream)
        e1.synchronize()
        return e0.elapsed_time(e1)

    for _ in range(warmup):
        one()
    s.synchronize()
    torch.cuda.synchronize()
    repeats = 1
    burst_ms = None
    if flush is None:
        # calibrate R on a first block of K steps so that the timed region is >= min_ms (same R on every rank);
        # that block, a few ms right after warm-up, is also the BURST figure: on B200 this kernel set slows by
        # 10-15 % after ~50 ms of back-to-back steps (sw_power_cap: the SM clock drops and the plane loop is
        # bound by SM latency, not by DRAM; a plain copy keeps 6.6 TB/s), so both are reported
        cal = block(steps)
        burst_ms = cal / steps
        repeats = max(1, int(np.ceil(min_ms / max(cal, 1e-3))))
        if dist is not None:
            t = torch.tensor([repeats], dtype=torch.int64, device=s.device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            repeats = int(t.item())
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    if flush is None:
        ms = block(steps * repeats) / repeats
    else:  # L2-resident workload: flush between timed steps, time each step by its own event pair
        evs = []
        for _ in range(steps):
            with torch.cuda.stream(s.stream):
                flush.zero_()
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            e0.record(s.stream)
            one()
            e1.record(s.stream)
            evs.append((e0, e1))
        s.synchronize()
        ms = sum(a.elapsed_time(b) for a, b in evs)
    torch.cuda.synchronize()
    sec = ms * 1e-3
    sec = max_over_ranks(torch, sec, dist, s.device)
    if dist is not None:
        dist.barrier()
    s.burst_ms_per_step = burst_ms
    return sec, s, repeats


def time_warm(torch, s, steps):
    """The same step back to back with nothing flushed in between (what hr_step(n) / hr_relax see on an
    L2-resident grid); seconds per step."""
    out2 = torch.zeros(2, dtype=torch.float64, device=s.device)
    for _ in range(5):
        s.hr_step_residual_async(0, out2)
    s.synchronize()
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    e0.record(s.stream)
    for _ in range(steps):
        s.hr_step_residual_async(0, out2)
    e1.record(s.stream)
    e1.synchronize()
    return e0.elapsed_time(e1) * 1e-3 / steps


def time_e2e(torch, s, steps, warmup, dist):
    """Same step through the C ABI with host buffers: H2D of (u, v) from pinned memory, the step,
    D2H of the residual.  Returns (seconds max over ranks, h2d bytes, d2h bytes)."""
    u = torch.zeros(s.ntot, dtype=s.tdtype).pin_memory()
    v = torch.zeros(s.ntot, dtype=s.tdtype).pin_memory()

    def one():
        s.hr_set_state_pinned(u, v)     # hr_set_state with host pointers: H2D + ghost fill
        s.hr_step(1)
        return s.hr_residual(0)         # D2H of {sum w H^2, sum w}, synchronises

    for _ in range(warmup):
        one()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    e0.record(s.stream)
    for _ in range(steps):
        one()
    e1.record(s.stream)
    e1.synchronize()
    sec = max(e0.elapsed_time(e1) * 1e-3, 0.0)
    wall = time.perf_counter() - t0
    sec = max(sec, wall) if wall > 0 else sec  # host-side marshalling counts too
    sec = max_over_ranks(torch, sec, dist, s.device)
    w = 8 if s.dtype == "f64" else 4
    return sec, 2 * s.ntot * w, 16


NOMINAL_HBM_GBS = 8000.0  # DGX B200 figure (7.7 TB/s HGX), context only (B200_PROFILING.md)


def flops_per_point(fd_order: int) -> int:
    """Algorithmic flops per interior point-substep: three second derivatives at
    3n + 1 and two first derivatives at 3n - 1 flops (n = NG, symmetric pairing), ~10 for the metric
    combination, ~25 for (psi + u)^-7 incl. one reciprocal, ~10 for k_u, c^2 and the RK combine."""
    n = fd_order // 2
    return 3 * (3 * n + 1) + 2 * (3 * n - 1) + 45


def roofline(s, prof_ms, peak, peak_src, fd_order, traffic, alu_peak):
    """Fused substep kernel, mean of the four stage launches.
      achieved / frac     SURVEY.md section 8(d): 10 w algorithmic bytes per interior point-substep (running-sum RK4:
                          8w, 12w, 12w, 8w) x N_int / mean launch duration -- kept so that rounds stay comparable
      moved / frac_moved  the bytes the shipped arrangement has to move: 8 w per point-substep in fp64 (ACC-free
                          RK4: 6w, 10w, 8w, 8w), 8.5 w in fp32 (its stage 4 also reads Y) -- THE distance to the roof
      traffic / frac_dram DRAM bytes per launch ncu measured on the committed capture (profiles/traffic.json)
      frac_nominal        moved bytes against the nominal 8 TB/s
      alu                 algorithmic flops per second against the FMA peak measured in this
                          run by hr_measure_alu_peak: shows which roof binds (HBM, by an order of magnitude)"""
    w = 8 if s.dtype == "f64" else 4
    mean_ms = sum(prof_ms[:4]) / 4.0
    sec = mean_ms * 1e-3
    bytes_per_launch = 10 * w * s.n_int
    moved = (8.0 if s.dtype == "f64" else 8.5) * w * s.n_int
    achieved = bytes_per_launch / sec / 1e9
    fl = flops_per_point(fd_order)
    out = {"bound": "hbm", "kernel": "fused substep k_march (RHS + radiation + RK combine + ghost images; stage 1 also "
                                      "reduces the residual), mean of the 4 stages",
           "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
           "peak_source": peak_src, "algorithmic_bytes_per_launch": bytes_per_launch,
           "moved_bytes_per_launch": moved, "moved_GBs": moved / sec / 1e9, "frac_moved": moved / sec / 1e9 / peak,
           "frac_nominal": moved / sec / 1e9 / NOMINAL_HBM_GBS, "peak_nominal": NOMINAL_HBM_GBS,
           "traffic": traffic, "frac_dram": (traffic / sec / 1e9 / peak) if traffic else None,
           "launch_ms": {"stage1": prof_ms[0], "stage2": prof_ms[1], "stage3": prof_ms[2],
                         "stage4": prof_ms[3], "inner_fill_x4": prof_ms[4], "residual": prof_ms[5]},
           "substep_kernel_share_of_step": sum(prof_ms[:4]) / sum(prof_ms),
           "alu": {"flops_per_point_substep": fl, "achieved_tflops": fl * s.n_int / sec / 1e12,
                   "peak_tflops": alu_peak, "frac": (fl * s.n_int / sec / 1e12 / alu_peak) if alu_peak else None,
                   "peak_source": "measured in this run (hr_measure_alu_peak: register-resident FMA chains)",
                   "arithmetic_intensity_flop_per_byte": fl / (moved / s.n_int),
                   "ridge_flop_per_byte": (alu_peak * 1e3 / peak) if alu_peak else None}}
    return out


def load_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(dtype):
    """dram bytes per launch of the fused kernel from the committed ncu --set full capture, if any."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(path) as f:
            return json.load(f).get(dtype)
    except (OSError, ValueError):
        return None


def run_many(args, name):
    """N independent grids on one GPU (the paper's Fig. 6 shape): hr_step_many = one CUDA graph with a branch per
    solver.  Host wall clock around `--steps` steps with a device synchronise on both sides (the call is host-driven:
    one graph replay per 8 steps), after `--warmup` x 8 steps; N = 1 is the sequential reference of the same call."""
    import torch
    import paper_2501_14030_b200 as hr
    out = {"metric": METRIC + ", N independent grids advanced together (hr_step_many)", "unit": UNIT,
           "n_solvers": args.many, "steps": args.steps, "config": {"workload": name}, "data": "synthetic"}
    for dtype in ("f64", "f32"):
        res = {}
        for n in sorted({1, args.many}):
            idx = int(name[5:].split(":")[0]) if name.startswith("sweep") else 0
            ps = [workload(name.replace(f"sweep{idx}", f"sweep{idx + i}", 1)) if name.startswith("sweep") else workload(name)
                  for i in range(n)]
            ss = [hr.Solver(q, dtype=dtype) for q in ps]
            hr.hr_step_many(ss, 8 * args.warmup)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            hr.hr_step_many(ss, args.steps)
            torch.cuda.synchronize()
            sec = time.perf_counter() - t0
            pts = ps[0]["n"][0] * ps[0]["n"][1] * ps[0]["n"][2]
            res[n] = {"us_per_grid_step": sec / args.steps / n * 1e6, "value": 4.0 * pts * n * args.steps / sec}
            for x in ss:
                x.close()
        out[dtype] = dict(res[args.many], vs_sequential=res[1]["us_per_grid_step"] / res[args.many]["us_per_grid_step"],
                          sequential_us_per_grid_step=res[1]["us_per_grid_step"])
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="config3")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--oracle-single", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--no-f32", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the extra config0/1/2 timings")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"],
                    help="precision of the headline leg (f32: for profiling the fp32 kernels alone)")
    ap.add_argument("--many", type=int, default=0, metavar="N",
                    help="row f2 instead of the headline line: N independent solvers of --workload advanced together by "
                         "hr_step_many (PAPER.md:337-347), --steps steps, both precisions; prints its own JSON line")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    name = args.workload
    p = workload(name)
    if args.many > 0:
        run_many(args, name)
        return

    if args.oracle_single:
        oracle_single(p, name)
        return
    if args.impl == "reference":
        run_reference(args, p, name)
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2501_14030_b200 as hr

    T = [x + p["fd_order"] for x in p["n"]]
    ntot = T[0] * T[1] * T[2]
    n_int = p["n"][0] * p["n"][1] * p["n"][2]
    flush_l2 = 10 * ntot * 8 <= 126e6  # fp64 working set fits L2 -> flush between timed steps
    peak, peak_src = load_peak()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    if args.dtype == "f32":
        args.no_f32 = True
        flush_l2 = 10 * ntot * 4 <= 126e6
    alu = {"f64": hr.hr_measure_alu_peak("f64", False, local),
           "f32": max(hr.hr_measure_alu_peak("f32", False, local), hr.hr_measure_alu_peak("f32", True, local))}
    sec64, s64, repeats = time_resident(torch, hr, p, args.dtype, args.steps, args.warmup, dist, flush_l2)
    launches_per_step = s64.launches_per_step  # the residual rides on the first substep's launch
    value = replicas_value(world, n_int, args.steps, sec64)
    burst = None
    if s64.burst_ms_per_step:
        w64 = 8 if args.dtype == "f64" else 4
        mv = (8.0 if args.dtype == "f64" else 8.5) * w64 * n_int * 4
        burst = {"what": f"the first {args.steps} steps after warm-up, timed alone ({s64.burst_ms_per_step * args.steps:.1f} ms): "
                         "before the power cap lowers the SM clock; `value` is the sustained figure",
                 "value": world * n_int * 4 / (s64.burst_ms_per_step * 1e-3), "ms_per_step": s64.burst_ms_per_step,
                 "frac_moved": mv / (s64.burst_ms_per_step * 1e-3) / 1e9 / peak}
    path = {"step_graph": s64.hr_query("step_graph"), "resid_graph": s64.hr_query("resid_graph"),
            "plan_zc": s64.hr_query("plan_zc"), "plan_items": s64.hr_query("plan_items"),
            "plan_grid": s64.hr_query("plan_grid")}

    prof64 = s64.hr_profile_step(min(max(args.steps, 20), 100), True)
    roof = roofline(s64, prof64, peak, peak_src, p["fd_order"], load_traffic(args.dtype), alu[args.dtype])
    sec_e2e, h2d, d2h = time_e2e(torch, s64, max(3, min(args.steps, 10)), 3, dist)
    e2e_steps = max(3, min(args.steps, 10))
    e2e = {"value": world * n_int * 4 * e2e_steps / sec_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "steps": e2e_steps,
           "what": "per step: hr_set_state(u, v from pinned host memory) + residual + 1 RK4 step + "
                   "residual read back to the host"}
    s64.close()
    del s64
    torch.cuda.empty_cache()

    f32 = None
    if not args.no_f32:
        sec32, s32, rep32 = time_resident(torch, hr, p, "f32", args.steps, args.warmup, dist,
                                          10 * ntot * 4 <= 126e6)
        prof32 = s32.hr_profile_step(min(max(args.steps, 20), 100), True)
        r32 = roofline(s32, prof32, peak, peak_src, p["fd_order"], load_traffic("f32"), alu["f32"])
        f32 = {"value": world * n_int * 4 * args.steps / sec32, "unit": UNIT,
               "ms_per_step": 1e3 * sec32 / args.steps, "repeats": rep32, "roofline": r32,
               "burst": {"value": world * n_int * 4 / (s32.burst_ms_per_step * 1e-3),
                         "ms_per_step": s32.burst_ms_per_step} if s32.burst_ms_per_step else None}
        s32.close()
        del s32

    # clocks over all timed legs (resident fp64, per-launch profile, e2e, fp32): the device is under load
    # throughout, and the headline region alone (K steps of < 1 ms) is shorter than a few samples
    clocks = sampler.stop() if rank == 0 else None

    # the smaller configs of BASELINE.json on the same box (rank 0, N = 1 only): L2-resident grids where
    # the step is bound by launch latency and the serial plane march, reported beside the headline
    also = None
    if world == 1 and args.workload == "config3" and not args.no_also:
        also = {}
        for other in ("config0", "config1", "config2"):
            po = workload(other)
            To = [x + po["fd_order"] for x in po["n"]]
            nto = To[0] * To[1] * To[2]
            nio = po["n"][0] * po["n"][1] * po["n"][2]
            entry = {"n_interior": list(po["n"]), "fd_order": po["fd_order"],
                     "l2": "L2 flushed between timed steps" if 10 * nto * 8 <= 126e6 else "larger than L2"}
            for dt, w in (("f64", 8), ("f32", 4)):
                sec, so, _ = time_resident(torch, hr, po, dt, 50, 5, None, 10 * nto * w <= 126e6)
                warm = time_warm(torch, so, 200)
                grid = so.hr_query("plan_grid")
                # the floor under a step of 4 dependent launches of this grid, whatever the kernels do
                floor_us = hr.hr_measure_launch_floor(4, int(grid), 128, 300, local)
                moved_w = 8.0 if dt == "f64" else 8.5
                entry[dt] = {"value": nio * 4 * 50 / sec, "unit": UNIT, "ms_per_step": 1e3 * sec / 50,
                             "warm_l2": {"value": nio * 4 / warm, "ms_per_step": 1e3 * warm,
                                         "what": "steps back to back, nothing flushed (hr_step(n), hr_relax)"},
                             "launch_floor_ms_per_step": 1e-3 * floor_us,
                             "floor_what": f"CUDA graph of 4 dependent empty launches, {grid} CTAs x 128 threads",
                             "frac_moved_warm": moved_w * w * nio * 4 / warm / 1e9 / peak,
                             "plan": {"zc": so.hr_query("plan_zc"), "items": so.hr_query("plan_items"),
                                      "grid": grid}}
                so.close()
                del so
            also[other] = entry

    if dist is not None:
        dist.barrier()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sec64 / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": config_dict(p, name, world), "clocks": clocks, "e2e": e2e,
            "gpu_launches": launches_per_step * args.steps * repeats, "repeats": repeats,
            "timed_region_ms": 1e3 * sec64 * repeats, "burst": burst, "roofline": roof, "f32": f32, "path": path,
            "library": hr.hr_version()}
    if also is not None:
        line["also"] = also
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(p, name)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
