"""Driver of the FMA ablation (Fig. 4): runs the paper-arrangement RHS
kernel (variant 1: one thread per point, block (32, NGHOSTS, 1), no shared memory, k stored in HBM) -- and, for
comparison, the fused marching kernel (variant 0) -- once each on a workload, so that ncu can count their
instruction mix:

    HR_B200_LIB=libhr_b200_nofmad.so ncu --metrics smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,... \\
        -k regex:'k_paper_rhs|k_march' python -m paper_2501_14030_b200.ablation --workload config3 --dtype f64

Product-side code: no oracle here (the accuracy half of the ablation is tests/test_gpu_ablation_fma.py).
"""
import argparse

import numpy as np


def main():
    import hr_workloads as W
    from . import Solver, binding
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="config3")
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    args = ap.parse_args()
    p = W.config(int(args.workload[6:]))
    rng_u, rng_v = W.random_state((p["n"][0] + p["fd_order"]) * (p["n"][1] + p["fd_order"])
                                  * (p["n"][2] + p["fd_order"]), seed=5)
    dt = np.float64 if args.dtype == "f64" else np.float32
    for variant in (1, 0):
        s = Solver(p, dtype=args.dtype, variant=variant)
        s.hr_set_state(rng_u.astype(dt), rng_v.astype(dt))
        s.hr_eval_rhs()
        s.synchronize()
        s.close()
    print("library:", binding.LIB_PATH)


if __name__ == "__main__":
    main()
