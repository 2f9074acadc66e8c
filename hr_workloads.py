"""Seeded, synthetic workloads shared by the oracle-side and CUDA-side tests and by bench.py.

This module holds NO arithmetic of the method (no stencils, metric factors, sources, maps): it
only names BASELINE.json's configurations as plain parameter dicts and draws seeded random
numbers.  Both `oracle.hr_oracle.Oracle(params)` and `paper_2501_14030_b200.Solver(params)`
take the same dict.  Values not fixed by BASELINE.json / PAPER.md (AMAX, SINHWAA, origin, eta,
c_min) are the readings C5, C6, C9, C10 listed in DESIGN.md.

Puncture row layout: [m, x, y, z, Px, Py, Pz, Sx, Sy, Sz].
"""
import numpy as np

SWEEP_SEED = 20250114  # seed + point index


def _base(**kw):
    d = dict(origin=(0.0, 0.0, 0.0), bscale=0.0, cfl=0.5, c_min=1.0)
    d.update(kw)
    return d


def config(i: int, scale: float = 1.0) -> dict:
    """BASELINE.json configs[i] for i in 0..3.  `scale` < 1 shrinks the grid (N2 kept even,
    every N_a >= NG) for the reduced cases the oracle finishes in seconds."""

    def sc(n, order):
        ng = order // 2
        out = [max(ng, int(round(x * scale))) for x in n]
        out[2] += out[2] % 2
        return tuple(out)

    if i == 0:
        return _base(name="config0", coord="SinhSpherical", n=sc((64, 16, 16), 4), fd_order=4,
                     amp=1.0e4, sinhw=0.2,
                     punctures=[[1.0, 0, 0, 0, 0, 0, 0, 0, 0, 0.2]], eta=2.0, steps=200)
    if i in (1, 2):
        n = (128, 64, 16) if i == 1 else (256, 128, 32)
        return _base(name=f"config{i}", coord="SinhSymTP", n=sc(n, 8), fd_order=8, amp=1.0e6,
                     sinhw=0.07, bscale=5.0,
                     punctures=[[0.5, 0, 0, +5.0, +0.0953, 0, 0, 0, 0, 0],
                                [0.5, 0, 0, -5.0, -0.0953, 0, 0, 0, 0, 0]],
                     eta=100.0 if i == 1 else 800.0, steps=2000)
    if i == 3:
        return _base(name="config3", coord="SinhSymTP", n=sc((512, 256, 64), 10), fd_order=10,
                     amp=1.0e6, sinhw=0.07, bscale=5.0, origin=(0.0, 0.0, -3.0),
                     punctures=[[0.8, 0, 0, +2.0, +0.08, 0, 0, 0.1, 0.05, 0.2],
                                [0.2, 0, 0, -8.0, -0.08, 0, 0, 0.0, 0.0, -0.02]],
                     eta=6400.0, steps=5000)
    raise ValueError(i)


SWEEP_GRIDS = [(64, 64, 64), (128, 128, 128), (256, 128, 64), (256, 256, 256), (512, 256, 128),
               (512, 256, 256)]


def random_punctures(seed: int, count: int = 2) -> list:
    """configs[4]: m ~ U(0.1,1), |P| < 0.2, |S| < 0.3 m^2 (uniform in the ball), on the z-axis
    with z ~ U(-10,10)."""
    rng = np.random.default_rng(seed)

    def in_ball(radius):
        while True:
            x = rng.uniform(-1.0, 1.0, 3)
            if x @ x < 1.0:
                return radius * x

    rows = []
    for _ in range(count):
        m = rng.uniform(0.1, 1.0)
        z = rng.uniform(-10.0, 10.0)
        P = in_ball(0.2)
        S = in_ball(0.3 * m * m)
        rows.append([m, 0.0, 0.0, z, *P, *S])
    return rows


def sweep_point(index: int, n, coord: str, fd_order: int) -> dict:
    """One point of configs[4]'s throughput sweep (grid x coordinate system x FD order)."""
    if coord in ("SinhSpherical", "SinhCylindrical", "SinhCartesian"):  # C24, C25: same amplitude and width
        geo = dict(amp=1.0e4, sinhw=0.2)
    else:
        geo = dict(amp=1.0e6, sinhw=0.07, bscale=5.0)
    return _base(name=f"sweep{index}", coord=coord, n=tuple(n), fd_order=fd_order,
                 punctures=random_punctures(SWEEP_SEED + index), eta=11.0, steps=100, **geo)


def random_state(ntot: int, seed: int, dtype=np.float64, amplitude: float = 0.1):
    """u, v ~ amplitude * U(-1,1) at every one of the ntot points (ghosts too; the caller makes
    them ghost-consistent with its own boundary map if it wants to)."""
    rng = np.random.default_rng(seed)
    u = amplitude * rng.uniform(-1.0, 1.0, ntot)
    v = amplitude * rng.uniform(-1.0, 1.0, ntot)
    return u.astype(dtype), v.astype(dtype)
