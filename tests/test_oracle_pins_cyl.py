"""Pins of the cylindrical-like reference metric (reading C24; PAPER.md:351 names the family,
nothing more): the oracle's SinhCylindrical branch checked against what the mathematics fixes, never against
itself -- the same pins P2, P3, P4, P8, P9, P11 the spherical-like systems have, each chosen so that a plausible
slip (a dropped first-derivative term, a wrong sign of the Z term, a transposed axis, a wrong one-sided stencil
on an end face) fails it.  CPU only (`-m "not gpu"`).
"""
import numpy as np
import pytest

from oracle import hr_oracle as O
from tests.test_oracle_pins import grid_cart, small, CID

CID["SinhCylindrical"] = 2
CYL = dict(coord="SinhCylindrical", amp=8.0, sinhw=0.5, bscale=0.0)


# P2c: round-trip map == closed-form integer map written independently (C14 for C24): x0-low ghosts
# reflect through the axis (rho -> -rho, phi + pi, z unchanged), phi wraps, everything beyond the outer
# cylinder or the end faces (with interior phi, x0 >= 0) is an outer point.
def closed_form_cyl(n, ng):
    N0, N1, N2 = n
    T0, T1, T2 = N0 + 2 * ng, N1 + 2 * ng, N2 + 2 * ng
    dst, src, outer = [], [], []
    for i2 in range(T2):
        for i1 in range(T1):
            for i0 in range(T0):
                in0, in1, in2 = ng <= i0 < N0 + ng, ng <= i1 < N1 + ng, ng <= i2 < N2 + ng
                if in0 and in1 and in2:
                    continue
                idx = i0 + T0 * (i1 + T1 * i2)
                if in2 and i0 >= ng and (i0 >= N0 + ng or not in1):
                    outer.append(idx)
                    continue
                j0, shift = i0, 0
                if i0 < ng:
                    j0, shift = 2 * ng - 1 - i0, 1
                j2 = (i2 - ng + shift * (N2 // 2)) % N2 + ng
                dst.append(idx)
                src.append(j0 + T0 * (i1 + T1 * j2))
    return np.array(dst, np.int32), np.array(src, np.int32), np.array(outer, np.int32)


@pytest.mark.parametrize("n,order", [((8, 6, 8), 4), ((6, 4, 4), 2), ((10, 8, 6), 8), ((12, 6, 10), 10)])
def test_p2c_roundtrip_map_equals_closed_form(n, order):
    o = O.Oracle(small(CYL, n, order))
    dst, src, outer = o.bc_lists()
    cd, cs, co = closed_form_cyl(n, order // 2)
    assert np.array_equal(dst, cd) and np.array_equal(src, cs) and np.array_equal(outer, co)
    assert o.bc_max_frac_err() < 1e-6
    assert not np.isin(src, dst).any()  # single hop
    ng = order // 2
    assert o.n_outer == ng * (n[1] + 2 * ng) * n[2] + 2 * ng * n[0] * n[2]
    assert o.n_inner + o.n_outer + n[0] * n[1] * n[2] == o.ntot
    # some inner sources are outer points (x0-low ghosts beyond an end face): outer first, then inner
    assert np.isin(src, outer).any()


def test_c8c_coordinates_and_outer_extent():
    o = O.Oracle(small(CYL, (8, 6, 8), 4))
    x0, x1, x2 = o.coords()
    assert x1[2] == pytest.approx(-1 + 1 / 6) and x1[-3] == pytest.approx(1 - 1 / 6)
    assert np.allclose(np.diff(x1), 2 / 6) and np.allclose(np.diff(x2), 2 * np.pi / 8)
    e = O.map_to_cart(2, 8.0, 0.5, 0.0, 1.0, -1.0, 0.0)
    assert e[0] == pytest.approx(8.0, rel=1e-13) and e[2] == pytest.approx(-8.0, rel=1e-13)
    rng = np.random.default_rng(5)
    for _ in range(50):
        a, b, p_ = rng.uniform(0.01, 1.2), rng.uniform(-1.2, 1.2), rng.uniform(-np.pi, np.pi - 1e-3)
        back = O.map_from_cart(2, 8.0, 0.5, 0.0, O.map_to_cart(2, 8.0, 0.5, 0.0, a, b, p_))
        assert np.allclose(back, [a, b, p_], rtol=0, atol=1e-9)


# P3c: Laplacian factors == generic Laplace-Beltrami of the coordinate map (sympy, 40 digits)
@pytest.mark.parametrize("ckw", [CYL, dict(coord="SinhCylindrical", amp=1.0e4, sinhw=0.2, bscale=0.0)])
def test_p3c_laplacian_factors_match_laplace_beltrami(ckw):
    sp = pytest.importorskip("sympy")
    import mpmath
    x0, x1, ph = sp.symbols("x0 x1 ph", real=True)
    amp, Wd = sp.Rational(str(ckw["amp"])), sp.Rational(str(ckw["sinhw"]))
    R = amp * sp.sinh(x0 / Wd) / sp.sinh(1 / Wd)
    Z = amp * sp.sinh(x1 / Wd) / sp.sinh(1 / Wd)
    X = sp.Matrix([R * sp.cos(ph), R * sp.sin(ph), Z])
    q = [x0, x1, ph]
    J = X.jacobian(q)
    g = sp.simplify(J.T * J)
    sqrtg = sp.sqrt(g[0, 0] * g[1, 1] * g[2, 2])
    second = [1 / g[a, a] for a in range(3)]
    first = [sp.diff(sqrtg / g[a, a], q[a]) / sqrtg for a in range(3)]
    f = sp.lambdify(q, [g[0, 1], g[0, 2], g[1, 2], *second, *first, sp.sqrt(g[0, 0]), sp.sqrt(g[1, 1]),
                        sp.sqrt(g[2, 2])], "mpmath")
    mpmath.mp.dps = 40
    rng = np.random.default_rng(3)
    for _ in range(12):
        a, b, p_ = rng.uniform(0.02, 1.0), rng.uniform(-1.0, 1.0), rng.uniform(-np.pi, np.pi)
        vals = [float(v) for v in f(mpmath.mpf(a), mpmath.mpf(b), mpmath.mpf(p_))]
        assert abs(vals[0]) < 1e-12 * vals[9] * vals[10]  # diagonal
        h, gf = O.metric_at(2, ckw["amp"], ckw["sinhw"], 0.0, a, b)
        assert np.allclose(h, vals[9:12], rtol=1e-12)
        assert np.allclose(gf[:3], vals[3:6], rtol=1e-12)
        assert gf[3] == pytest.approx(vals[6], rel=1e-10, abs=1e-12 * abs(vals[3]))
        assert gf[4] == pytest.approx(vals[7], rel=1e-10, abs=1e-12 * abs(vals[4]))  # the -Z''/Z'^3 term
        assert abs(vals[8]) < 1e-10 * abs(vals[5])  # no u_2 term, nothing depends on phi


# P4c: discrete Laplacian of an off-centre Gaussian converges at the nominal order; a harmonic polynomial
def _lap_error(n, order, func, lapfunc, ckw):
    p = small(ckw, n, order)
    o = O.Oracle(p)
    xyz = grid_cart(o, p)
    lap = o.laplacian(func(xyz))
    m = o.interior_mask()
    w = np.broadcast_to(o.planes()["w"][None], (o.T[2], o.T[1], o.T[0])).reshape(-1)
    err = (lap - lapfunc(xyz))[m]
    return np.sqrt(np.sum(w[m] * err**2) / np.sum(w[m])) / np.sqrt(np.sum(w[m] * lapfunc(xyz)[m] ** 2) / np.sum(w[m]))


@pytest.mark.parametrize("order", [4, 8])
def test_p4c_laplacian_converges_at_nominal_order(order):
    ckw = dict(coord="SinhCylindrical", amp=2.0, sinhw=0.8, bscale=0.0)
    xc, sig = np.array([0.3, -0.2, 0.25]), 0.9

    def f(x):
        return np.exp(-np.sum((x - xc) ** 2, axis=1) / sig**2)

    def lf(x):
        d2 = np.sum((x - xc) ** 2, axis=1)
        return (4 * d2 / sig**4 - 6 / sig**2) * f(x)

    n = (12, 24, 24) if order == 4 else (16, 32, 32)
    e1 = _lap_error(n, order, f, lf, ckw)
    e2 = _lap_error(tuple(2 * k for k in n), order, f, lf, ckw)
    rate = np.log2(e1 / e2)
    assert e2 < e1 and rate > order - 0.6, (e1, e2, rate)


def test_p4c_harmonic_polynomial_is_annihilated():
    p = small(dict(coord="SinhCylindrical", amp=4.0, sinhw=0.6, bscale=0.0), (24, 32, 16), 8)
    o = O.Oracle(p)
    x, y, z = grid_cart(o, p).T
    m = o.interior_mask()
    lap = o.laplacian(x**2 - y**2 + 3 * x * z - 2 * z)[m]
    one = o.laplacian(z**2)[m]  # = 2 up to truncation: exercises u_11 and the -Z''/Z'^3 u_1 term alone
    assert np.median(np.abs(one - 2.0)) < 2e-2
    assert np.median(np.abs(lap)) < 2e-2 * np.median(np.abs(one))


# P8c: ds = min_a |h_a| dx^a from a numerical Jacobian; Courant number == CFL everywhere
def test_p8c_cfl_identity_and_dt_bruteforce():
    n, order = (16, 12, 8), 4
    p = small(CYL, n, order, cfl=0.4)
    o = O.Oracle(p)
    pl = o.planes()
    ng = order // 2
    x0, x1, _ = o.coords()
    dx = [1 / n[0], 2 / n[1], 2 * np.pi / n[2]]
    ds = np.zeros((o.T[1], o.T[0]))
    for j in range(o.T[1]):
        for i in range(o.T[0]):
            q = np.array([x0[i], x1[j], 0.37])
            vals = []
            for a in range(3):
                e = np.zeros(3)
                e[a] = 1e-6
                d = (O.map_to_cart(2, p["amp"], p["sinhw"], 0.0, *(q + e))
                     - O.map_to_cart(2, p["amp"], p["sinhw"], 0.0, *(q - e))) / 2e-6
                vals.append(np.linalg.norm(d) * dx[a])
            ds[j, i] = min(vals)
    assert np.allclose(pl["ds"], ds, rtol=1e-6)
    assert o.dsmin == pytest.approx(ds[ng:-ng, ng:-ng].min(), rel=1e-6)
    assert o.dt == pytest.approx(0.4 * o.dsmin, rel=1e-15)
    assert np.allclose(pl["c"] * o.dt / pl["ds"], 0.4, rtol=1e-13)


# P9c: the exact outgoing wave G(r - t)/r is annihilated at second order on the outer cylinder AND on both end
# faces (backward / forward one-sided stencils along x1), corners included; with the pulse on an end face the Z
# term carries most of d_r f, so a wrong sign or a wrong one-sided stencil there is an O(1) error.
@pytest.mark.parametrize("centre", [8.5, 10.5])
def test_p9c_outgoing_wave_is_annihilated_at_second_order(centre):
    ckw = dict(coord="SinhCylindrical", amp=8.0, sinhw=0.6, bscale=0.0)

    def G(r):
        return np.exp(-((r - centre) / 2.0) ** 2)

    def dG(r):
        return -2 * (r - centre) / 4.0 * G(r)

    errs, face_errs = [], []
    for n in ((24, 48, 8), (48, 96, 8)):
        p = small(ckw, n, 4)
        o = O.Oracle(p)
        xyz = grid_cart(o, p)
        r = np.linalg.norm(xyz, axis=1)
        f = G(r) / r
        ku, kv = o.rhs(f, 2 * f, part="outer")
        _, _, outer = o.bc_lists()
        c = np.broadcast_to(o.planes()["c"][None], (o.T[2], o.T[1], o.T[0])).reshape(-1)
        exact = -c * dG(r) / r
        scale = np.max(np.abs(exact[outer]))
        errs.append(np.max(np.abs(ku[outer] - exact[outer])) / scale)
        assert np.allclose(kv[outer], 2 * ku[outer], rtol=1e-13, atol=1e-15 * scale)
        rest = np.ones(o.ntot, bool)
        rest[outer] = False
        assert not ku[rest].any() and not kv[rest].any()
        # the end faces alone (interior x0): low face uses the forward stencil, high face the backward one
        T0, T1 = o.T[0], o.T[1]
        i0, i1 = outer % T0, (outer // T0) % T1
        ng = 2
        for face in (i1 < ng, i1 >= n[1] + ng):
            sel = outer[face & (i0 < n[0] + ng)]
            face_errs.append(np.max(np.abs(ku[sel] - exact[sel])) / scale)
    assert errs[0] < 0.3 and errs[1] < 0.08 and errs[1] < errs[0] / 3.0, errs
    assert face_errs[2] < face_errs[0] / 3.0 and face_errs[3] < face_errs[1] / 3.0, face_errs
    assert abs(face_errs[2] - face_errs[3]) < 1e-6 * max(face_errs[2:])  # the two faces mirror each other


# P6c / P11c: zero momentum and spin is an exact fixed point; the residual decays monotonically after transients
def test_p6c_p11c_fixed_point_and_decay():
    punct0 = [[0.5, 0, 0, 1.0, 0, 0, 0, 0, 0, 0], [0.5, 0, 0, -1.0, 0, 0, 0, 0, 0, 0]]
    ckw = dict(coord="SinhCylindrical", amp=1.0e3, sinhw=0.15, bscale=0.0)
    o = O.Oracle(small(ckw, (16, 32, 8), 4, punctures=punct0))
    z = np.zeros(o.ntot)
    u, v = o.step(z, z, 5)
    assert not u.any() and not v.any()
    punct = [[0.5, 0, 0, 1.0, 0.1, 0, 0, 0, 0, 0.05], [0.5, 0, 0, -1.0, -0.1, 0, 0, 0, 0, 0]]
    o = O.Oracle(small(ckw, (24, 48, 8), 6, punctures=punct, eta=4.0))
    psi, _ = o.source()
    u, v = z[:0], None
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
    dst, src, _ = o.bc_lists()
    assert np.array_equal(u[dst], u[src]) and np.array_equal(v[dst], v[src])  # C15 holds here too
