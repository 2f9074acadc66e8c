"""GPU parity at BASELINE.json's stated sizes and step counts (`-m gpu`): configs 0-3 stepped for their
full 200 / 2000 / 2000 / 5000 RK4 steps and configs[4]'s sweep grids at full size, compared with the
anchors the CPU oracle wrote on a CPU box (tests/golden/full_*.txt|npz, written by
tests/golden/make_golden_full.py from oracle/ only).  PAPER.md:254, 266 (section 5.1, Fig. 1): the paper's own
consistency claim is about agreement "halfway through relaxation" and "at the end of relaxation".

FROZEN BARS (a bar changes only in a commit that touches no kernel and names the reading):
  fp64 residual   |r_gpu - r_or| <= 1e-10 * max_n r_or(n)                      (C21 ii, every mark)
                  |r_gpu - r_or| <= 1e-10 * r_or   while r_or >= 1e-2 * max_n r_or(n)   (north_star, literal)
  fp64 state      max|u_gpu - u_or| <= 1e-10 * max|u_or| on the sampled points; v against |v| + eta |u|
  fp32 residual   |r_gpu32 - r_or64| <= 1e-4 * max_n r_or64(n)                 (asserted where
                  BASELINE.json asks for fp32, i.e. config 2, and on config 0, at every mark; everywhere as
                  envelopes: the GPU's largest miss over the run <= max(1e-4 * peak, 1.5 x the fp32 ORACLE's
                  largest miss over the run) -- two fp32 roundings of the same run are two noise samples)
  fp32 state      max|u_gpu32 - u_or64| <= 1.5 * max|u_or32 - u_or64| + 4 eps32 max|u|   (C21 iii: the GPU's
                  fp32 path may not drift more than 1.5x what the fp32 oracle itself drifts)
Every literal relative number is printed beside the fp32 oracle's own and written to
$HR_PARITY_OUT (default gpurun_out/) as parity_<case>_<dtype>.txt; BASELINE.md section 4 is that table.
"""
import os

import numpy as np
import pytest

import hr_workloads as W

pytestmark = pytest.mark.gpu

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
OUT = os.environ.get("HR_PARITY_OUT", os.path.join(os.path.dirname(os.path.dirname(GOLD)), "gpurun_out"))
EPS32 = float(np.finfo(np.float32).eps)
# The literal 1e-10 is asserted while the residual is within two decades of the run's largest one (C21 ii): the
# absolute error of the norm stays near kappa * eps * peak with kappa ~ 1e2 ... 1e3 after thousands of steps
# (measured: 7e-13 of peak at step 4500 of config 3, 7e-14 at step 800 of config 1), so the LITERAL relative
# number crosses 1e-10 once the residual has fallen 2-4 decades (1.7e-10 at 4e-3 of peak on config 3, 5.5e-10
# at 1.3e-4 on config 1) without any implementation being wrong; the state agrees to 2e-14 throughout.
LITERAL_DECADES = 1e-2


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2501_14030_b200 as pkg
    return pkg


def load(case):
    txt = os.path.join(GOLD, f"full_{case}.txt")
    if not os.path.exists(txt):
        pytest.skip(f"{txt} not written yet (python tests/golden/make_golden_full.py {case})")
    rows = np.loadtxt(txt, ndmin=2)
    return rows, np.load(os.path.join(GOLD, f"full_{case}.npz"))


def emit(case, dtype, lines):
    text = "\n".join(lines)
    print(text)
    try:
        os.makedirs(OUT, exist_ok=True)
        with open(os.path.join(OUT, f"parity_{case}_{dtype}.txt"), "w") as f:
            f.write(text + "\n")
    except OSError:
        pass


def sampled(s, idx):
    return s.hr_get_u()[idx].astype(np.float64), s.hr_get_v()[idx].astype(np.float64)


FULL = ["config0", "config1", "config2", "config3"]


@pytest.mark.parametrize("case", FULL)
def test_full_config_fp64(hr, case):
    rows, z = load(case)
    p = W.config(int(case[-1]))
    s = hr.Solver(p, dtype="f64")
    idx = z["idx"]
    peak = [rows[:, 1].max(), rows[:, 2].max()]
    lines = [f"# {case} fp64: n = {tuple(p['n'])}, fd_order {p['fd_order']}, eta {p['eta']}",
             "# step mode r_gpu r_oracle literal_rel rel_to_peak r_or/peak"]
    done = 0
    bad = []
    dst, src, _ = s.hr_get_bc_lists()
    for row in rows:
        m = int(row[0])
        s.hr_step(m - done)
        done = m
        for mode in (0, 1):
            r, ro = s.hr_residual(mode), row[1 + mode]
            lit, rel = abs(r - ro) / ro, abs(r - ro) / peak[mode]
            lines.append(f"{m} {mode} {r:.15e} {ro:.15e} {lit:.2e} {rel:.2e} {ro / peak[mode]:.1e}")
            if rel > 1e-10 or (ro >= LITERAL_DECADES * peak[mode] and lit > 1e-10):
                bad.append((m, mode, r, ro, lit, rel))
        if f"u64_{m}" in z:
            u, v = sampled(s, idx)
            ou, ov = z[f"u64_{m}"], z[f"v64_{m}"]
            eu = np.abs(u - ou).max() / np.abs(ou).max()
            ev = np.abs(v - ov).max() / (np.abs(ov).max() + p["eta"] * np.abs(ou).max())
            lines.append(f"# step {m}: sampled state ({idx.size} points incl. outer and inner ghosts) "
                         f"max|du|/max|u| {eu:.2e}  max|dv|/(max|v| + eta max|u|) {ev:.2e}")
            if eu > 1e-10 or ev > 1e-10:
                bad.append((m, "state", eu, ev))
    uf = s.hr_get_u()
    emit(case, "f64", lines)
    assert not bad, (case, bad)
    assert np.array_equal(uf[dst], uf[src])  # C15: ghosts bitwise equal to their sources
    s.close()


@pytest.mark.parametrize("case", FULL)
def test_full_config_fp32(hr, case):
    rows, z = load(case)
    rows = rows[~np.isnan(rows[:, 3])]  # the marks the fp32 oracle ran to
    p = W.config(int(case[-1]))
    s = hr.Solver(p, dtype="f32")
    idx = z["idx"]
    lines = [f"# {case} fp32 vs the fp64 oracle: n = {tuple(p['n'])}, fd_order {p['fd_order']}, eta {p['eta']}",
             "# step mode r_gpu32 r_oracle64 gpu32_literal_rel oracle32_literal_rel gpu32_rel_to_peak "
             "oracle32_rel_to_peak"]
    strict = case in ("config0", "config2")  # BASELINE.json: fp32 is asked for on config 2 (and the sweep)
    done = 0
    bad = []
    peak = [0.0, 0.0]
    floor = [0.0, 0.0]
    miss = [0.0, 0.0]
    for row in rows:
        m = int(row[0])
        s.hr_step(m - done)
        done = m
        for mode in (0, 1):
            ro, r32o = row[1 + mode], row[3 + mode]
            peak[mode] = max(peak[mode], ro)  # C21: max over n <= N of r_or64(n), n = 0 included
            r = s.hr_residual(mode)
            dg, do = abs(r - ro), abs(r32o - ro)
            lines.append(f"{m} {mode} {r:.9e} {ro:.9e} {dg / ro:.2e} {do / ro:.2e} {dg / peak[mode]:.2e} "
                         f"{do / peak[mode]:.2e}")
            if strict and dg > 1e-4 * peak[mode]:
                bad.append((m, mode, r, ro, r32o, dg / peak[mode]))
            floor[mode] = max(floor[mode], do)  # envelopes over the run: the fp32 oracle's largest miss
            miss[mode] = max(miss[mode], dg)    # and the GPU's
        if f"u32_{m}" in z:
            u, v = sampled(s, idx)
            ou, ov = z[f"u64_{m}"], z[f"v64_{m}"]
            eg, eo = np.abs(u - ou).max(), np.abs(z[f"u32_{m}"].astype(np.float64) - ou).max()
            umax = np.abs(ou).max()
            lines.append(f"# step {m}: sampled fp32 state vs fp64 oracle: gpu {eg / umax:.2e}  fp32 oracle "
                         f"{eo / umax:.2e}  (of max|u|)")
            if eg > 1.5 * eo + 4 * EPS32 * umax:
                bad.append((m, "state", eg / umax, eo / umax))
    for mode in (0, 1):
        lines.append(f"# mode {mode}: largest miss over the run, of the peak residual: gpu32 "
                     f"{miss[mode] / peak[mode]:.2e}  fp32 oracle {floor[mode] / peak[mode]:.2e}")
        if miss[mode] > max(1e-4 * peak[mode], 1.5 * floor[mode]):
            bad.append(("envelope", mode, miss[mode] / peak[mode], floor[mode] / peak[mode]))
    emit(case, "f32", lines)
    assert not bad, (case, bad)
    s.close()


def sweep_cases():
    k = 0
    for n in W.SWEEP_GRIDS:
        for coord in ("SinhSpherical", "SinhSymTP"):
            for order in (4, 10):
                yield k, n, coord, order
                k += 1


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_sweep_grids_full_size_rhs(hr, dtype):
    """configs[4]: one RHS evaluation (hr_eval_rhs, all N_tot entries written) on every sweep grid at full
    size, both coordinate systems, orders 4 and 10, against the oracle's k on a fixed sample of interior,
    outer and inner-ghost points; bars 1e-12 (fp64) / 1e-5 (fp32), max-norm relative per field (C21 i)."""
    path = os.path.join(GOLD, "full_config4.npz")
    if not os.path.exists(path):
        pytest.skip("full_config4.npz not written yet")
    z = np.load(path)
    tol = 1e-12 if dtype == "f64" else 1e-5
    lines = [f"# configs[4] {dtype}: per-RHS max-norm relative error on the sampled points (bar {tol:g})",
             "# k grid coord order err_ku err_kv"]
    for k, n, coord, order in sweep_cases():
        p = W.sweep_point(k, n, coord, order)
        s = hr.Solver(p, dtype=dtype)
        u, v = W.random_state(s.ntot, seed=1000 + k)  # hr_set_state makes it ghost-consistent (C14)
        if dtype == "f32":
            u, v = u.astype(np.float32), v.astype(np.float32)
        s.hr_set_state(u, v)
        ku, kv = s.hr_eval_rhs()
        idx = z[f"idx_{k}"]
        tag = "32in" if dtype == "f32" else ""
        oku, okv = z[f"ku{tag}_{k}"], z[f"kv{tag}_{k}"]
        kmax = z[f"kmax_{k}"][2:] if dtype == "f32" else z[f"kmax_{k}"][:2]
        eu = np.abs(ku[idx].astype(np.float64) - oku).max() / kmax[0]
        ev = np.abs(kv[idx].astype(np.float64) - okv).max() / kmax[1]
        lines.append(f"{k} {n[0]}x{n[1]}x{n[2]} {coord} {order} {eu:.2e} {ev:.2e}")
        assert eu <= tol and ev <= tol, (k, n, coord, order, eu, ev)
        s.close()
        del ku, kv, u, v
    emit("config4", dtype, lines)


def f3_cases():
    k = 200
    for n in [(128, 128, 128), (256, 128, 64)]:
        for coord in ("SinhCylindrical", "SinhCartesian"):
            for order in (4, 10):
                yield k, n, coord, order
                k += 1


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_f3_reference_metrics_at_sweep_sizes(hr, dtype):
    """The cylindrical-like and Cartesian-like systems (readings C24 / C25) at two sweep sizes, orders 4 and 10: one
    RHS evaluation against the oracle's k on 8192 sampled points each (interior, the outer points of every face,
    inner ghosts where the system has them); same bars as configs[4]."""
    path = os.path.join(GOLD, "full_f3.npz")
    if not os.path.exists(path):
        pytest.skip("full_f3.npz not written yet (python tests/golden/make_golden_full.py f3)")
    z = np.load(path)
    tol = 1e-12 if dtype == "f64" else 1e-5
    lines = [f"# f3 grids {dtype}: per-RHS max-norm relative error on the sampled points (bar {tol:g})",
             "# k grid coord order err_ku err_kv"]
    for k, n, coord, order in f3_cases():
        p = W.sweep_point(k, n, coord, order)
        s = hr.Solver(p, dtype=dtype)
        u, v = W.random_state(s.ntot, seed=1000 + k)
        if dtype == "f32":
            u, v = u.astype(np.float32), v.astype(np.float32)
        s.hr_set_state(u, v)
        ku, kv = s.hr_eval_rhs()
        idx = z[f"idx_{k}"]
        tag = "32in" if dtype == "f32" else ""
        kmax = z[f"kmax_{k}"][2:] if dtype == "f32" else z[f"kmax_{k}"][:2]
        eu = np.abs(ku[idx].astype(np.float64) - z[f"ku{tag}_{k}"]).max() / kmax[0]
        ev = np.abs(kv[idx].astype(np.float64) - z[f"kv{tag}_{k}"]).max() / kmax[1]
        lines.append(f"{k} {n[0]}x{n[1]}x{n[2]} {coord} {order} {eu:.2e} {ev:.2e}")
        assert eu <= tol and ev <= tol, (k, n, coord, order, eu, ev)
        s.close()
    emit("f3", dtype, lines)
