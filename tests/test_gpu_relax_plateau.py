"""f1 (Alg. 1 l.8-18): the relaxation driver run to its plateau on
BASELINE.json configs[0] and configs[1] -- hr_relax with a stopping tolerance, the residual history (both norms)
tabulated, the plateau compared with the CPU oracle's at the same step counts, and the wall time to tolerance.

The residual is that of the DISCRETE equation, so its floor is the rounding level of H (eps * sum|terms|), not the
truncation error of the grid: the history falls geometrically until it meets that floor and stays there.  Once on
the floor the norm is a sum of rounding errors and two correct implementations agree in order of magnitude only;
above it (within LIVE of the floor) they agree to the C21 (ii) bar.  The table goes to $HR_PARITY_OUT (default
gpurun_out/) as relax_<config>.txt; profiles/r2_relax.md is a copy."""
import os
import time

import numpy as np
import pytest

import hr_workloads as W
from oracle.hr_oracle import Oracle

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
OUT = os.environ.get("HR_PARITY_OUT", os.path.join(ROOT, "gpurun_out"))

CASES = [("config0", 0, 4000, 100), ("config1", 1, 8000, 200)]


@pytest.mark.parametrize("name,idx,max_steps,every", CASES, ids=[c[0] for c in CASES])
def test_relax_to_the_plateau(name, idx, max_steps, every):
    import paper_2501_14030_b200 as hr
    p = W.config(idx)
    hist = {}
    for mode in (0, 1):
        s = hr.Solver(p, residual_mode=mode)
        t0 = time.perf_counter()
        done, res, h = s.hr_relax(max_steps, every, 0.0, mode)
        wall = time.perf_counter() - t0
        assert done == max_steps and len(h) == max_steps // every + 1 and res == h[-1]
        hist[mode] = (np.asarray(h), wall)
        s.close()
    # the plateau: the level the last quarter of the history sits on
    lines = [f"# {name}: hr_relax(max_steps = {max_steps}, check_every = {every}, tol = 0), fp64, n = {tuple(p['n'])}, "
             f"order {p['fd_order']}, eta {p['eta']}",
             f"# wall time of {max_steps} steps incl. {max_steps // every + 1} residual checks: "
             f"mode 0 {hist[0][1] * 1e3:.1f} ms, mode 1 {hist[1][1] * 1e3:.1f} ms "
             f"({hist[1][1] / max_steps * 1e6:.1f} us per step)",
             "# step  gpu_mode0  gpu_mode1  oracle_mode0  oracle_mode1  rel0  rel1"]
    o = Oracle(p)
    ou, ov = np.zeros(o.ntot), np.zeros(o.ntot)
    marks = sorted(set(list(range(0, max_steps + 1, max_steps // 8))))
    ref, at = {}, 0
    for m in marks:
        ou, ov = o.step(ou, ov, m - at)
        at = m
        ref[m] = (o.residual(ou, 0), o.residual(ou, 1))
    bad = []
    for mode in (0, 1):
        h = hist[mode][0]
        floor = np.median(h[-len(h) // 4:])
        peak = h.max()
        assert floor < 1e-6 * peak, (name, mode, floor, peak)           # it did relax by six decades
        assert h[-1] < 3.0 * floor and np.all(h[-len(h) // 4:] < 10 * floor)  # and it stays on the floor
        for m in marks:
            g, r = h[m // every], ref[m][mode]
            if r > 100.0 * floor:  # above the rounding floor: the C21 (ii) bar
                if abs(g - r) > 1e-10 * peak:
                    bad.append((mode, m, g, r))
            elif not (0.1 < g / r < 10.0):  # on the floor: same order of magnitude
                bad.append((mode, m, g, r, "floor"))
        hist[mode] = (h, hist[mode][1], floor, peak)
    for k in range(0, max_steps // every + 1):
        m = k * every
        g0, g1 = hist[0][0][k], hist[1][0][k]
        if m in ref:
            r0, r1 = ref[m]
            lines.append(f"{m} {g0:.6e} {g1:.6e} {r0:.6e} {r1:.6e} {abs(g0 - r0) / r0:.1e} {abs(g1 - r1) / r1:.1e}")
        else:
            lines.append(f"{m} {g0:.6e} {g1:.6e}")
    for mode in (0, 1):
        h, wall, floor, peak = hist[mode]
        k = int(np.argmax(h < 10 * floor))
        lines.append(f"# mode {mode}: peak {peak:.3e}, floor {floor:.3e} ({floor / peak:.1e} of the peak), reached "
                     f"(within 10x) after {k * every} steps = {wall * k * every / max_steps * 1e3:.1f} ms")
    text = "\n".join(lines)
    print(text)
    try:
        os.makedirs(OUT, exist_ok=True)
        with open(os.path.join(OUT, f"relax_{name}.txt"), "w") as f:
            f.write(text + "\n")
    except OSError:
        pass
    assert not bad, bad
