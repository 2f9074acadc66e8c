"""Writes the full-size, full-length anchors of BASELINE.json's configs 0-4 from the CPU oracle ONLY
(never the CUDA path): tests/golden/full_<case>.txt (residual histories, text) and
tests/golden/full_<case>.npz (sampled u, v / k).  The GPU parity tests compare hr_step + hr_residual +
sampled hr_get_u / hr_eval_rhs against these files (tests/test_gpu_full_configs.py).

    python tests/golden/make_golden_full.py config0 config1 config2 config3 config4

The paper prints no value of u or ||H|| (PAPER.md:254, 266 only state that CPU and GPU agree at
t_mid and t_end), so these are not paper values: they are what the pinned oracle (P1-P14,
tests/test_oracle_pins.py) computes for the inputs of hr_workloads.py at their stated sizes and step
counts ("parity unpinned" outputs, oracle/hr_oracle.h).  The oracle's results do not depend on the
thread count (static loops, per-plane residual partials added in a fixed order).

Text file columns (one row per mark):
  steps  r64_mode0 r64_mode1  r32_mode0 r32_mode1  r32state_in64_mode0 r32state_in64_mode1  max|u64|
where r64 = fp64 oracle; r32 = fp32 oracle, fp32 state evaluated by the fp32 residual; r32state_in64 =
the fp32 oracle's state evaluated by the fp64 residual (C21: separates state drift from evaluation
noise).  fp32 columns are nan where the fp32 oracle was not run.

npz: idx (int64 public flat indices: interior, outer and inner-ghost samples), and for each sample
mark m: u64_m, v64_m (and u32_m, v32_m).  config4: per grid, coordinate system and order, the sampled
k_u, k_v of one RHS evaluation of a seeded random ghost-consistent state.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import hr_workloads as W  # noqa: E402
from oracle.hr_oracle import Oracle, num_threads  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
SAMPLE_SEED = 250114030

# case -> (params, residual marks, sample marks, last step of the fp32 oracle)
CASES = {
    "config0": (lambda: W.config(0), list(range(0, 201, 20)), [100, 200], 200),
    "config1": (lambda: W.config(1), list(range(0, 2001, 100)), [1000, 2000], 2000),
    "config2": (lambda: W.config(2), list(range(0, 2001, 100)), [1000, 2000], 2000),
    "config3": (lambda: W.config(3), [0, 50, 500, 1000, 1500, 2000, 2500, 3000, 3500, 4000, 4500, 5000],
                [50, 500, 2500, 5000], 500),
}


def sample_indices(o, seed, n_interior=8192, n_outer=2048, n_inner=2048):
    """Fixed sample of public flat indices: interior, outer and inner-ghost points."""
    rng = np.random.default_rng(seed)
    dst, _, outer = o.bc_lists()
    interior = np.flatnonzero(o.interior_mask())
    pick = lambda a, n: np.sort(rng.choice(a, size=min(n, a.size), replace=False))  # noqa: E731
    return np.concatenate([pick(interior, n_interior), pick(outer, n_outer), pick(dst, n_inner)]).astype(np.int64)


def run_case(name):
    make, marks, smarks, last32 = CASES[name]
    p = make()
    t0 = time.time()
    o = Oracle(p)
    idx = sample_indices(o, SAMPLE_SEED + int(name[-1]))
    u, v = np.zeros(o.ntot), np.zeros(o.ntot)
    u32, v32 = u.astype(np.float32), v.astype(np.float32)
    arrays = {"idx": idx}
    rows = []
    done = 0
    for m in marks:
        u, v = o.step(u, v, m - done)
        run32 = m <= last32
        if run32:
            u32, v32 = o.step(u32, v32, m - done)
        done = m
        nan = float("nan")
        r32 = [o.residual(u32, k) for k in (0, 1)] if run32 else [nan, nan]
        r3264 = [o.residual(u32.astype(np.float64), k) for k in (0, 1)] if run32 else [nan, nan]
        rows.append((m, o.residual(u, 0), o.residual(u, 1), *r32, *r3264, float(np.abs(u).max())))
        print(name, rows[-1], "%.0f s" % (time.time() - t0), flush=True)
        if m in smarks:
            arrays[f"u64_{m}"], arrays[f"v64_{m}"] = u[idx], v[idx]
            if run32:
                arrays[f"u32_{m}"], arrays[f"v32_{m}"] = u32[idx], v32[idx]
    with open(os.path.join(HERE, f"full_{name}.txt"), "w") as f:
        f.write(f"# written by tests/golden/make_golden_full.py from oracle/ only ({num_threads()} threads, "
                f"{time.time() - t0:.0f} s); see its docstring for the columns\n")
        f.write(f"# {name}: n = {tuple(p['n'])}, fd_order = {p['fd_order']}, eta = {p['eta']}, dt = {o.dt:.17e}\n")
        for r in rows:
            f.write("%d " % r[0] + " ".join("%.17e" % x for x in r[1:]) + "\n")
    np.savez_compressed(os.path.join(HERE, f"full_{name}.npz"), **arrays)


# configs[4]: one RHS evaluation per (grid, coordinate system, order) at full size, sampled
SWEEP_ORDERS = (4, 10)


def sweep_cases():
    k = 0
    for n in W.SWEEP_GRIDS:
        for coord in ("SinhSpherical", "SinhSymTP"):
            for order in SWEEP_ORDERS:
                yield k, n, coord, order
                k += 1


def run_sweep():
    arrays = {}
    t0 = time.time()
    for k, n, coord, order in sweep_cases():
        p = W.sweep_point(k, n, coord, order)
        o = Oracle(p)
        idx = sample_indices(o, SAMPLE_SEED + 100 + k, 4096, 1024, 1024)
        u, v = W.random_state(o.ntot, seed=1000 + k)
        u, v = o.apply_inner(u), o.apply_inner(v)
        ku, kv = o.rhs(u, v)
        # fp32 inputs: the same state rounded once; the arithmetic reference stays the fp64 oracle
        u32, v32 = u.astype(np.float32), v.astype(np.float32)
        ku32, kv32 = o.rhs(u32.astype(np.float64), v32.astype(np.float64))
        tag = f"{k}"
        arrays[f"idx_{tag}"] = idx
        arrays[f"ku_{tag}"], arrays[f"kv_{tag}"] = ku[idx], kv[idx]
        arrays[f"ku32in_{tag}"], arrays[f"kv32in_{tag}"] = ku32[idx], kv32[idx]
        arrays[f"kmax_{tag}"] = np.array([np.abs(ku).max(), np.abs(kv).max(), np.abs(ku32).max(), np.abs(kv32).max()])
        print("config4", k, n, coord, order, "%.0f s" % (time.time() - t0), flush=True)
        del o, u, v, ku, kv, ku32, kv32
    np.savez_compressed(os.path.join(HERE, "full_config4.npz"), **arrays)


# f3 (readings C24 / C25): the cylindrical-like and Cartesian-like systems at sweep sizes, same recipe
F3_GRIDS = [(128, 128, 128), (256, 128, 64)]


def f3_cases():
    k = 200
    for n in F3_GRIDS:
        for coord in ("SinhCylindrical", "SinhCartesian"):
            for order in SWEEP_ORDERS:
                yield k, n, coord, order
                k += 1


def run_f3():
    arrays = {}
    t0 = time.time()
    for k, n, coord, order in f3_cases():
        p = W.sweep_point(k, n, coord, order)
        o = Oracle(p)
        idx = sample_indices(o, SAMPLE_SEED + k, 4096, 2048, 1024) if o.n_inner > 0 else np.sort(
            np.random.default_rng(SAMPLE_SEED + k).choice(o.ntot, size=8192, replace=False)).astype(np.int64)
        u, v = W.random_state(o.ntot, seed=1000 + k)
        u, v = o.apply_inner(u), o.apply_inner(v)
        ku, kv = o.rhs(u, v)
        u32, v32 = u.astype(np.float32), v.astype(np.float32)
        ku32, kv32 = o.rhs(u32.astype(np.float64), v32.astype(np.float64))
        arrays[f"idx_{k}"] = idx
        arrays[f"ku_{k}"], arrays[f"kv_{k}"] = ku[idx], kv[idx]
        arrays[f"ku32in_{k}"], arrays[f"kv32in_{k}"] = ku32[idx], kv32[idx]
        arrays[f"kmax_{k}"] = np.array([np.abs(ku).max(), np.abs(kv).max(), np.abs(ku32).max(), np.abs(kv32).max()])
        print("f3", k, n, coord, order, "%.0f s" % (time.time() - t0), flush=True)
    np.savez_compressed(os.path.join(HERE, "full_f3.npz"), **arrays)


if __name__ == "__main__":
    for name in sys.argv[1:]:
        if name == "config4":
            run_sweep()
        elif name == "f3":
            run_f3()
        else:
            run_case(name)
