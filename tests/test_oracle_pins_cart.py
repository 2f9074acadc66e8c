"""Pins of the Cartesian-like reference metric (reading C25; PAPER.md:351 names the family, nothing
more): the oracle's SinhCartesian branch against what the mathematics fixes -- P2, P3, P4, P8, P9, P6/P11 as for
the other systems.  What is new here and must be caught: a u_2 term and an x2-dependent u_22 factor, a wave speed
and a volume weight that depend on all three coordinates, outer points on all six faces (edges and corners
included) with one-sided stencils along every axis, and no inner points at all.  CPU only (`-m "not gpu"`).
"""
import numpy as np
import pytest

from oracle import hr_oracle as O
from tests.test_oracle_pins import grid_cart, small, CID

CID["SinhCartesian"] = 3
CART = dict(coord="SinhCartesian", amp=8.0, sinhw=0.5, bscale=0.0)


@pytest.mark.parametrize("n,order", [((8, 6, 8), 4), ((6, 4, 4), 2), ((10, 8, 6), 8), ((7, 9, 6), 6)])
def test_p2k_every_ghost_point_is_an_outer_point(n, order):
    o = O.Oracle(small(CART, n, order))
    dst, src, outer = o.bc_lists()
    assert dst.size == 0 and src.size == 0 and o.n_inner == 0
    m = o.interior_mask()
    assert np.array_equal(outer, np.flatnonzero(~m).astype(np.int32))  # ascending, all ghosts, nothing else
    assert o.n_outer + n[0] * n[1] * n[2] == o.ntot
    x0, x1, x2 = o.coords()
    ng = order // 2
    for x, k in ((x0, n[0]), (x1, n[1]), (x2, n[2])):
        assert x[ng] == pytest.approx(-1 + 1 / k) and x[-ng - 1] == pytest.approx(1 - 1 / k)
        assert np.allclose(np.diff(x), 2 / k)
    rng = np.random.default_rng(5)
    for _ in range(30):
        q = rng.uniform(-1.2, 1.2, 3)
        back = O.map_from_cart(3, 8.0, 0.5, 0.0, O.map_to_cart(3, 8.0, 0.5, 0.0, *q))
        assert np.allclose(back, q, rtol=0, atol=1e-9)
    assert np.allclose(O.map_to_cart(3, 8.0, 0.5, 0.0, 1.0, -1.0, 1.0), [8.0, -8.0, 8.0], rtol=1e-13)


@pytest.mark.parametrize("ckw", [CART, dict(coord="SinhCartesian", amp=1.0e4, sinhw=0.2, bscale=0.0)])
def test_p3k_laplacian_factors_match_laplace_beltrami(ckw):
    """All six factors (u_00, u_11, u_22, u_0, u_1, u_2) and the three scale factors against the generic
    orthogonal-coordinates formula from the coordinate map, sympy at 40 digits; the x2 ones come out of the
    grid object (axis2), evaluated at its own x2 coordinates."""
    sp = pytest.importorskip("sympy")
    import mpmath
    q = sp.symbols("x0 x1 x2", real=True)
    amp, Wd = sp.Rational(str(ckw["amp"])), sp.Rational(str(ckw["sinhw"]))
    X = sp.Matrix([amp * sp.sinh(t / Wd) / sp.sinh(1 / Wd) for t in q])
    J = X.jacobian(q)
    g = J.T * J
    sqrtg = sp.sqrt(g[0, 0] * g[1, 1] * g[2, 2])
    second = [1 / g[a, a] for a in range(3)]
    first = [sp.diff(sqrtg / g[a, a], q[a]) / sqrtg for a in range(3)]
    f = sp.lambdify(q, [*second, *first, sp.sqrt(g[0, 0]), sp.sqrt(g[1, 1]), sp.sqrt(g[2, 2]), g[0, 1], g[0, 2],
                        g[1, 2]], "mpmath")
    mpmath.mp.dps = 40
    o = O.Oracle(small(ckw, (6, 6, 8), 4))
    _, _, x2 = o.coords()
    ax = o.axis2()
    rng = np.random.default_rng(3)
    for k in range(12):
        a, b = rng.uniform(-1.0, 1.0, 2)
        c = x2[k % x2.size]
        vals = [float(v) for v in f(mpmath.mpf(a), mpmath.mpf(b), mpmath.mpf(float(c)))]
        assert vals[9] == vals[10] == vals[11] == 0.0
        h, gf = O.metric_at(3, ckw["amp"], ckw["sinhw"], 0.0, a, b)
        assert np.allclose(h[:2], vals[6:8], rtol=1e-12)
        assert np.allclose(gf[:2], vals[0:2], rtol=1e-12)
        assert gf[3] == pytest.approx(vals[3], rel=1e-10) and gf[4] == pytest.approx(vals[4], rel=1e-10)
        i = k % x2.size
        assert ax["zh"][i] == pytest.approx(vals[8], rel=1e-12)
        assert ax["z22"][i] == pytest.approx(vals[2], rel=1e-12)
        assert ax["z2"][i] == pytest.approx(vals[5], rel=1e-10)
        assert ax["zds"][i] == pytest.approx(vals[8] * 2 / 8, rel=1e-12)  # h2 dx2, N2 = 8


def _lap_error(n, order, func, lapfunc, ckw):
    p = small(ckw, n, order)
    o = O.Oracle(p)
    xyz = grid_cart(o, p)
    lap = o.laplacian(func(xyz))
    m = o.interior_mask()
    w2 = o.planes()["w"][None] * o.axis2()["zh"][:, None, None]
    w = w2.reshape(-1)
    err = (lap - lapfunc(xyz))[m]
    return np.sqrt(np.sum(w[m] * err**2) / np.sum(w[m])) / np.sqrt(np.sum(w[m] * lapfunc(xyz)[m] ** 2) / np.sum(w[m]))


@pytest.mark.parametrize("order", [4, 8])
def test_p4k_laplacian_converges_at_nominal_order(order):
    ckw = dict(coord="SinhCartesian", amp=2.0, sinhw=0.8, bscale=0.0)
    xc, sig = np.array([0.3, -0.2, 0.25]), 0.9

    def f(x):
        return np.exp(-np.sum((x - xc) ** 2, axis=1) / sig**2)

    def lf(x):
        d2 = np.sum((x - xc) ** 2, axis=1)
        return (4 * d2 / sig**4 - 6 / sig**2) * f(x)

    n = (16, 18, 20) if order == 4 else (24, 26, 28)
    e1 = _lap_error(n, order, f, lf, ckw)
    e2 = _lap_error(tuple(2 * k for k in n), order, f, lf, ckw)
    rate = np.log2(e1 / e2)
    assert e2 < e1 and rate > order - 0.6, (e1, e2, rate)


def test_p4k_each_axis_term_alone_and_a_harmonic_polynomial():
    p = small(dict(coord="SinhCartesian", amp=4.0, sinhw=0.6, bscale=0.0), (32, 30, 28), 8)
    o = O.Oracle(p)
    x, y, z = grid_cart(o, p).T
    m = o.interior_mask()
    for t in (x, y, z):  # lap(t^2) = 2: exercises u_aa and the -X''/X'^3 u_a term of each axis on its own
        assert np.median(np.abs(o.laplacian(t**2)[m] - 2.0)) < 2e-2
    lap = o.laplacian(x**2 - y**2 + 3 * x * z - 2 * z + y * z)[m]
    assert np.median(np.abs(lap)) < 4e-2


def test_p8k_spacing_wave_speed_and_time_step():
    n, order = (8, 10, 12), 4  # the finest spacing is along x2: ds_min must see it
    p = small(CART, n, order, cfl=0.4, punctures=[[1.0, 0.1, 0.2, 0.3, 0.1, 0, 0, 0, 0, 0.1]])
    o = O.Oracle(p)
    ng = order // 2
    x0, x1, x2 = o.coords()
    dx = [2 / n[0], 2 / n[1], 2 / n[2]]
    pl, ax = o.planes(), o.axis2()
    ds3 = np.zeros((o.T[2], o.T[1], o.T[0]))
    for k in range(o.T[2]):
        for j in range(o.T[1]):
            for i in range(o.T[0]):
                q = np.array([x0[i], x1[j], x2[k]])
                vals = []
                for a in range(3):
                    e = np.zeros(3)
                    e[a] = 1e-6
                    d = (O.map_to_cart(3, p["amp"], p["sinhw"], 0.0, *(q + e))
                         - O.map_to_cart(3, p["amp"], p["sinhw"], 0.0, *(q - e))) / 2e-6
                    vals.append(np.linalg.norm(d) * dx[a])
                ds3[k, j, i] = min(vals)
    ds_or = np.minimum(pl["ds"][None], ax["zds"][:, None, None])
    assert np.allclose(ds_or, ds3, rtol=1e-6)
    assert o.dsmin == pytest.approx(ds3[ng:-ng, ng:-ng, ng:-ng].min(), rel=1e-6)
    assert o.dt == pytest.approx(0.4 * o.dsmin, rel=1e-15)
    # the wave speed the RHS uses: k_v = c^2 (lap u + S psi^-7); with u = 0, v = 0: k_v / (S psi^-7) = c^2
    z = np.zeros(o.ntot)
    _, kv = o.rhs(z, z, part="interior")
    psi, S = o.source()
    m = o.interior_mask()
    c2 = kv[m] / (S[m] * psi[m] ** -7.0)
    assert np.allclose(np.sqrt(c2) * o.dt / ds3.reshape(-1)[m], 0.4, rtol=1e-10)


@pytest.mark.parametrize("centre", [8.5, 11.0])
def test_p9k_outgoing_wave_is_annihilated_on_all_six_faces(centre):
    ckw = dict(coord="SinhCartesian", amp=8.0, sinhw=0.6, bscale=0.0)

    def G(r):
        return np.exp(-((r - centre) / 2.5) ** 2)

    def dG(r):
        return -2 * (r - centre) / 6.25 * G(r)

    errs, faces = [], []
    for n in ((24, 26, 28), (48, 52, 56)):
        p = small(ckw, n, 4)
        o = O.Oracle(p)
        xyz = grid_cart(o, p)
        r = np.linalg.norm(xyz, axis=1)
        f = G(r) / r
        ku, kv = o.rhs(f, 2 * f, part="outer")
        _, _, outer = o.bc_lists()
        # c at every point: c_min min(ds plane, zds) / ds_min
        c = (np.minimum(o.planes()["ds"][None], o.axis2()["zds"][:, None, None]) / o.dsmin).reshape(-1)
        exact = -c * dG(r) / r
        scale = np.max(np.abs(exact[outer]))
        errs.append(np.max(np.abs(ku[outer] - exact[outer])) / scale)
        assert np.allclose(kv[outer], 2 * ku[outer], rtol=1e-13, atol=1e-15 * scale)
        assert not ku[o.interior_mask()].any()
        T0, T1 = o.T[0], o.T[1]
        idx = [outer % T0, (outer // T0) % T1, outer // (T0 * T1)]
        ng = 2
        row = []
        for a in range(3):
            others = np.ones(outer.size, bool)
            for b in range(3):
                if b != a:
                    others &= (idx[b] >= ng) & (idx[b] < n[b] + ng)
            for side in (idx[a] < ng, idx[a] >= n[a] + ng):
                sel = outer[side & others]
                row.append(np.max(np.abs(ku[sel] - exact[sel])) / scale)
        faces.append(row)
    assert errs[0] < 0.3 and errs[1] < 0.08 and errs[1] < errs[0] / 3.0, errs
    for lo, hi in zip(faces[0], faces[1]):  # every face on its own converges at second order
        assert hi < lo / 3.0, faces
    for a in range(3):  # the low and the high face of an axis mirror each other
        assert abs(faces[1][2 * a] - faces[1][2 * a + 1]) < 1e-6 * max(faces[1])


def test_p6k_p11k_fixed_point_and_decay():
    punct0 = [[0.5, 0.1, 0, 1.0, 0, 0, 0, 0, 0, 0], [0.5, 0, 0.1, -1.0, 0, 0, 0, 0, 0, 0]]
    ckw = dict(coord="SinhCartesian", amp=1.0e3, sinhw=0.15, bscale=0.0)
    o = O.Oracle(small(ckw, (16, 16, 16), 4, punctures=punct0))
    z = np.zeros(o.ntot)
    u, v = o.step(z, z, 5)
    assert not u.any() and not v.any()
    punct = [[0.5, 0, 0, 1.0, 0.1, 0, 0, 0, 0, 0.05], [0.5, 0, 0, -1.0, -0.1, 0, 0, 0, 0, 0]]
    o = O.Oracle(small(ckw, (24, 24, 24), 6, punctures=punct, eta=0.5))  # eta dt = 0.35 (C10)
    psi, _ = o.source()
    u = np.zeros(o.ntot)
    v = np.zeros(o.ntot)
    hist = []
    for _ in range(16):
        u, v = o.step(u, v, 50)
        hist.append(o.residual(u, 1))
        assert np.all(psi + u > 0)
    h = np.array(hist)
    assert np.all(np.isfinite(h)) and np.all(np.diff(h[4:]) < 0), h
    assert h[-1] < 0.3 * h[4]
    # mode 0 weights |h0 h1 h2|: brute force from H
    r0, H = o.residual(u, 0, return_H=True)
    m = o.interior_mask()
    w = (o.planes()["w"][None] * o.axis2()["zh"][:, None, None]).reshape(-1)
    assert r0 == pytest.approx(np.sqrt(np.sum(w[m] * H[m] ** 2) / np.sum(w[m])), rel=1e-12)
