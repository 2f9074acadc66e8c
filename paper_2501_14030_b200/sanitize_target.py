"""Small driver for compute-sanitizer: the library's calls on three small grids -- BASELINE.json
configs[0], a ragged 10th-order SinhSymTP grid and the minimal 5x5x6 grid -- through hr_set_state, hr_eval_rhs,
hr_step(3), hr_step_residual_async, hr_relax, hr_residual, hr_get_u, hr_step_many, in both precisions.

    compute-sanitizer --tool memcheck|racecheck|initcheck python -m paper_2501_14030_b200.sanitize_target

Product-side code: no oracle; it only has to run clean.  Prints one line per case and "sanitize target done".
"""
import numpy as np


def main():
    import torch

    import hr_workloads as W
    from . import Solver, hr_step_many

    cases = [("config0", W.config(0)),
             ("tp_o10_ragged", W.sweep_point(2, (33, 21, 12), "SinhSymTP", 10)),
             ("minimal_o10", W.sweep_point(6, (5, 5, 6), "SinhSymTP", 10))]
    for name, p in cases:
        for dtype in ("f64", "f32"):
            s = Solver(p, dtype=dtype)
            u, v = W.random_state(s.ntot, seed=3, amplitude=1e-3)
            npdt = np.float64 if dtype == "f64" else np.float32
            s.hr_set_state(u.astype(npdt), v.astype(npdt))
            ku, kv = s.hr_eval_rhs()
            # step from u = v = 0 (C17): white noise is amplified ~7x per step on the 5-point grid and would
            # (rightly) end in HR_ERR_NUMERIC
            s.hr_set_state(np.zeros(s.ntot, npdt), np.zeros(s.ntot, npdt))
            # (the 5-point grid is not a stable discretisation: it gets one step of each kind, the others a few)
            few = 1 if name == "minimal_o10" else 3
            s.hr_step(few)
            out2 = torch.zeros(2, dtype=torch.float64, device=s.device)
            s.hr_step_residual_async(0, out2)
            s.synchronize()
            done, res, hist = s.hr_relax(2 * few - 1, few, 0.0, 1)
            r = s.hr_residual(0)
            uu = s.hr_get_u()
            t = Solver(p, dtype=dtype)
            hr_step_many([s, t], 1 if name == "minimal_o10" else 9)
            s.synchronize()
            t.synchronize()
            print(f"{name} {dtype}: |k_u| {np.abs(ku).max():.3e} residual {r:.6e} relax steps {done} "
                  f"history {len(hist)} max|u| {np.abs(uu).max():.3e}", flush=True)
            s.close()
            t.close()
    print("sanitize target done")


if __name__ == "__main__":
    main()
