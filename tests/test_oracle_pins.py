"""Pins P1-P14 (SURVEY.md Sec. 8c / DESIGN.md): the CPU oracle checked against what the paper and
the mathematics fix -- closed forms, invariants, textbook identities, brute force -- never
against itself.  CPU only (`-m "not gpu"`).
"""
from fractions import Fraction

import numpy as np
import pytest

import hr_workloads as W
from oracle import hr_oracle as O

SPH = dict(coord="SinhSpherical", amp=1.0e4, sinhw=0.2, bscale=0.0)
TP = dict(coord="SinhSymTP", amp=1.0e6, sinhw=0.07, bscale=5.0)
CID = {"SinhSpherical": 0, "SinhSymTP": 1}


def small(coord_kw, n, order, punctures=None, **kw):
    p = dict(origin=(0.0, 0.0, 0.0), cfl=0.5, c_min=1.0, eta=2.0, n=n, fd_order=order,
             punctures=punctures if punctures is not None else [[1.0, 0, 0, 0.3, 0, 0, 0, 0, 0, 0]])
    p.update(coord_kw)
    p.update(kw)
    return p


def grid_cart(o, p):
    """Cartesian coordinates of every grid point (ghosts included) via the oracle's own map,
    plus origin; shape (ntot, 3)."""
    x0, x1, x2 = o.coords()
    out = np.zeros((o.T[2], o.T[1], o.T[0], 3))
    for k, c in enumerate(x2):
        for j, b in enumerate(x1):
            for i, a in enumerate(x0):
                out[k, j, i] = O.map_to_cart(CID[p["coord"]], p["amp"], p["sinhw"], p["bscale"],
                                             a, b, c)
    return out.reshape(-1, 3) + np.asarray(p["origin"])


# ------------------------------------------------------------------------------------------
# P1  FD tables (C11): closed form == exact-rational Vandermonde solve; exact on polynomials
# ------------------------------------------------------------------------------------------
def exact_weights(n, deriv):
    """Solve sum_k w_k k^p = p! delta_{p,deriv}, p = 0..2n, over offsets -n..n, in rationals."""
    offs = list(range(-n, n + 1))
    m = len(offs)
    A = [[Fraction(k) ** p for k in offs] + [Fraction(1 if p == deriv else 0) * (1 if deriv < 2 else 2)]
         for p in range(m)]
    for col in range(m):  # Gauss-Jordan in exact arithmetic
        piv = next(r for r in range(col, m) if A[r][col] != 0)
        A[col], A[piv] = A[piv], A[col]
        A[col] = [x / A[col][col] for x in A[col]]
        for r in range(m):
            if r != col and A[r][col] != 0:
                A[r] = [x - A[r][col] * y for x, y in zip(A[r], A[col])]
    return {k: A[i][m] for i, k in enumerate(offs)}


@pytest.mark.parametrize("order", [2, 4, 6, 8, 10, 12])
def test_p1_fd_weights_equal_vandermonde(order):
    n = order // 2
    c1, d2 = O.fd_weights(order)
    w1, w2 = exact_weights(n, 1), exact_weights(n, 2)
    assert c1[0] == 0.0
    for k in range(1, n + 1):
        assert c1[k] == pytest.approx(float(w1[k]), rel=4e-16, abs=0)
        assert -c1[k] == pytest.approx(float(w1[-k]), rel=4e-16, abs=0)
        assert d2[k] == pytest.approx(float(w2[k]), rel=4e-16, abs=0)
        assert w2[k] == w2[-k]
    assert d2[0] == pytest.approx(float(w2[0]), rel=4e-16, abs=0)


def test_p1_known_low_order_tables():
    # textbook values (e.g. Fornberg 1988, Table 1)
    c1, d2 = O.fd_weights(2)
    assert np.allclose(c1, [0, 0.5], rtol=0, atol=0) and np.allclose(d2, [-2, 1], rtol=0, atol=0)
    c1, d2 = O.fd_weights(4)
    assert np.allclose(c1, [0, 2 / 3, -1 / 12], rtol=1e-16)
    assert np.allclose(d2, [-5 / 2, 4 / 3, -1 / 12], rtol=1e-16)
    c1, d2 = O.fd_weights(6)
    assert np.allclose(c1, [0, 3 / 4, -3 / 20, 1 / 60], rtol=1e-15)
    assert np.allclose(d2, [-49 / 18, 3 / 2, -3 / 20, 1 / 90], rtol=1e-15)


@pytest.mark.parametrize("order", [4, 6, 8, 10])
def test_p1_polynomial_exactness(order):
    n = order // 2
    c1, d2 = O.fd_weights(order)
    x = np.arange(-n, n + 1, dtype=np.float64)
    for p in range(0, order + 2):
        f = (x / n) ** p  # keep values O(1)
        first = sum(c1[k] * (f[n + k] - f[n - k]) for k in range(1, n + 1))
        second = d2[0] * f[n] + sum(d2[k] * (f[n + k] + f[n - k]) for k in range(1, n + 1))
        if p <= order:
            assert first == pytest.approx((1.0 / n) if p == 1 else 0.0, abs=2e-14)
        assert second == pytest.approx((2.0 / n**2) if p == 2 else 0.0, abs=2e-13)


# ------------------------------------------------------------------------------------------
# P2  grid + inner map (C8, C14): generic round trip == closed-form integer map, counts, one hop
# ------------------------------------------------------------------------------------------
def closed_form_inner_map(coord, n, ng):
    """The integer statement of C14, written independently of the oracle's fp64 round trip."""
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
                if i0 >= N0 + ng and in1 and in2:
                    outer.append(idx)
                    continue
                j0, j1, shift = i0, i1, 0
                if i0 < ng:  # r -> -r
                    j0 = 2 * ng - 1 - i0
                    shift += 1
                    if coord == "SinhSpherical":
                        j1 = T1 - 1 - j1  # theta -> pi - theta
                if j1 < ng:  # theta -> -theta
                    j1 = 2 * ng - 1 - j1
                    shift += 1
                elif j1 >= N1 + ng:  # theta -> 2 pi - theta
                    j1 = 2 * (N1 + ng) - 1 - j1
                    shift += 1
                j2 = (i2 - ng + (shift % 2) * (N2 // 2)) % N2 + ng
                dst.append(idx)
                src.append(j0 + T0 * (j1 + T1 * j2))
    return np.array(dst, np.int32), np.array(src, np.int32), np.array(outer, np.int32)


MAP_CASES = [(SPH, (8, 6, 8), 4), (SPH, (6, 4, 4), 2), (TP, (8, 6, 8), 4), (TP, (10, 8, 6), 8),
             (TP, (12, 6, 10), 10), (SPH, (64, 16, 16), 4)]


@pytest.mark.parametrize("ckw,n,order", MAP_CASES)
def test_p2_roundtrip_map_equals_closed_form(ckw, n, order):
    o = O.Oracle(small(ckw, n, order))
    dst, src, outer = o.bc_lists()
    cd, cs, co = closed_form_inner_map(ckw["coord"], n, order // 2)
    assert np.array_equal(dst, cd) and np.array_equal(src, cs) and np.array_equal(outer, co)
    assert o.bc_max_frac_err() < 1e-6
    assert np.all(np.diff(dst) > 0) and np.all(np.diff(outer) > 0)
    # single hop: no source is itself an inner ghost
    assert not np.isin(src, dst).any()
    # every point is exactly one of interior / outer / inner
    ng = order // 2
    assert o.n_outer == ng * n[1] * n[2]
    assert o.n_inner + o.n_outer + n[0] * n[1] * n[2] == o.ntot


def test_p2_counts_at_baseline_configs():
    # SURVEY.md Sec. 8 point-count table
    o0 = O.Oracle(W.config(0))
    assert (o0.ntot, o0.n_int, o0.n_outer, o0.n_inner) == (27200, 16384, 512, 10304)
    _, src, outer = o0.bc_lists()
    assert int(np.isin(src, outer).sum()) == 288  # C14: sources that are outer points
    o1 = O.Oracle(W.config(1))
    assert (o1.ntot, o1.n_int, o1.n_outer, o1.n_inner) == (235008, 131072, 4096, 99840)


def test_c8_cell_centred_coordinates():
    o = O.Oracle(small(SPH, (8, 6, 8), 4))
    x0, x1, x2 = o.coords()
    ng = 2
    assert x0[ng] == pytest.approx(0.5 / 8) and x0[-ng - 1] == pytest.approx(1 - 0.5 / 8)
    assert x1[ng] == pytest.approx(0.5 * np.pi / 6) and x2[ng] == pytest.approx(-np.pi + np.pi / 8)
    assert np.allclose(np.diff(x0), 1 / 8) and np.allclose(np.diff(x1), np.pi / 6)
    assert np.allclose(np.diff(x2), 2 * np.pi / 8)
    # mirror symmetry of ghosts about the faces (what makes the inner map close on grid points)
    assert np.allclose(x0[:ng], -x0[2 * ng - 1:ng - 1:-1])
    assert np.allclose(x1[:ng], -x1[2 * ng - 1:ng - 1:-1])


# ------------------------------------------------------------------------------------------
# P3  reference-metric factors (C4): generic Laplace-Beltrami from the coordinate map (sympy)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ckw", [dict(coord="SinhSpherical", amp=3.0, sinhw=0.4, bscale=0.0),
                                 dict(coord="SinhSymTP", amp=7.0, sinhw=0.3, bscale=1.7), SPH, TP])
def test_p3_laplacian_factors_match_laplace_beltrami(ckw):
    sp = pytest.importorskip("sympy")
    x0, th, ph = sp.symbols("x0 th ph", real=True)
    amp, Wd, b = sp.Rational(str(ckw["amp"])), sp.Rational(str(ckw["sinhw"])), sp.Rational(str(ckw["bscale"]))
    rho = amp * sp.sinh(x0 / Wd) / sp.sinh(1 / Wd)
    if ckw["coord"] == "SinhSpherical":
        X = sp.Matrix([rho * sp.sin(th) * sp.cos(ph), rho * sp.sin(th) * sp.sin(ph), rho * sp.cos(th)])
    else:
        X = sp.Matrix([rho * sp.sin(th) * sp.cos(ph), rho * sp.sin(th) * sp.sin(ph),
                       sp.sqrt(rho**2 + b**2) * sp.cos(th)])
    q = [x0, th, ph]
    J = X.jacobian(q)
    g = J.T * J
    sqrtg = sp.sqrt(g[0, 0] * g[1, 1] * g[2, 2])
    # lap u = (1/sqrt g) d_a( sqrt g g^{aa} d_a u ) for a diagonal metric
    second = [1 / g[a, a] for a in range(3)]
    first = [sp.diff(sqrtg / g[a, a], q[a]) / sqrtg for a in range(3)]
    f = sp.lambdify(q, [g[0, 1], g[0, 2], g[1, 2], *second, *first, sp.sqrt(g[0, 0]),
                        sp.sqrt(g[1, 1]), sp.sqrt(g[2, 2])], "mpmath")
    import mpmath
    mpmath.mp.dps = 40
    rng = np.random.default_rng(3)
    for _ in range(12):
        a, t, p_ = rng.uniform(0.02, 1.0), rng.uniform(0.05, np.pi - 0.05), rng.uniform(-np.pi, np.pi)
        vals = [float(v) for v in f(mpmath.mpf(a), mpmath.mpf(t), mpmath.mpf(p_))]
        scale = vals[9] * vals[10]
        assert abs(vals[0]) < 1e-12 * scale and abs(vals[1]) < 1e-12 * scale  # diagonal metric
        h, gf = O.metric_at(CID[ckw["coord"]], ckw["amp"], ckw["sinhw"], ckw["bscale"], a, t)
        assert np.allclose(h, vals[9:12], rtol=1e-12)
        assert np.allclose(gf[:3], vals[3:6], rtol=1e-12)            # u_00 u_11 u_22
        assert gf[3] == pytest.approx(vals[6], rel=1e-10, abs=1e-12 * abs(vals[3]))  # u_0
        assert gf[4] == pytest.approx(vals[7], rel=1e-10, abs=1e-12 * abs(vals[4]))  # u_1
        assert abs(vals[8]) < 1e-10 * abs(vals[5])                   # no u_2 term


def test_p3_symtp_reduces_to_spherical_for_small_b():
    for a, t in [(0.3, 0.7), (0.9, 2.1)]:
        hs, gs = O.metric_at(0, 5.0, 0.3, 0.0, a, t)
        ht, gt = O.metric_at(1, 5.0, 0.3, 1e-9, a, t)
        assert np.allclose(hs, ht, rtol=1e-12) and np.allclose(gs, gt, rtol=1e-12)


def test_c4_map_roundtrip_and_parity_images():
    rng = np.random.default_rng(5)
    for cid, kw in ((0, SPH), (1, TP)):
        for _ in range(50):
            a, t, p_ = rng.uniform(0.01, 1.1), rng.uniform(0.01, np.pi - 0.01), rng.uniform(-np.pi, np.pi - 1e-3)
            xyz = O.map_to_cart(cid, kw["amp"], kw["sinhw"], kw["bscale"], a, t, p_)
            back = O.map_from_cart(cid, kw["amp"], kw["sinhw"], kw["bscale"], xyz)
            assert np.allclose(back, [a, t, p_], rtol=0, atol=1e-9)
        # SymTP foci at z = +-b: A -> 0 on the axis
        if cid == 1:
            z = O.map_to_cart(1, kw["amp"], kw["sinhw"], kw["bscale"], 1e-12, 1e-9, 0.3)
            assert z[2] == pytest.approx(kw["bscale"], rel=1e-12)
        # outer radius = AMP at x0 = 1, theta = pi/2
        e = O.map_to_cart(cid, kw["amp"], kw["sinhw"], kw["bscale"], 1.0, np.pi / 2, 0.0)
        assert e[0] == pytest.approx(kw["amp"], rel=1e-13)


# ------------------------------------------------------------------------------------------
# P4  discrete Laplacian (C11, C12): analytic functions of the Cartesian coordinates
# ------------------------------------------------------------------------------------------
def _lap_error(ckw, n, order, func, lapfunc):
    p = small(ckw, n, order)
    o = O.Oracle(p)
    xyz = grid_cart(o, p)
    u = func(xyz)
    lap = o.laplacian(u)
    m = o.interior_mask()
    w = np.broadcast_to(o.planes()["w"][None], (o.T[2], o.T[1], o.T[0])).reshape(-1)
    err = (lap - lapfunc(xyz))[m]
    l2 = np.sqrt(np.sum(w[m] * err**2) / np.sum(w[m]))
    ref = np.sqrt(np.sum(w[m] * lapfunc(xyz)[m] ** 2) / np.sum(w[m]))
    return l2 / ref


@pytest.mark.parametrize("ckw", [dict(coord="SinhSpherical", amp=2.0, sinhw=0.8, bscale=0.0),
                                 dict(coord="SinhSymTP", amp=2.0, sinhw=0.8, bscale=0.6)])
@pytest.mark.parametrize("order", [4, 8])
def test_p4_laplacian_converges_at_nominal_order(ckw, order):
    xc, sig = np.array([0.3, -0.2, 0.25]), 0.9

    def f(x):
        return np.exp(-np.sum((x - xc) ** 2, axis=1) / sig**2)

    def lf(x):
        d2 = np.sum((x - xc) ** 2, axis=1)
        return (4 * d2 / sig**4 - 6 / sig**2) * f(x)

    n = (12, 12, 24) if order == 4 else (16, 16, 32)
    e1 = _lap_error(ckw, n, order, f, lf)
    e2 = _lap_error(ckw, tuple(2 * k for k in n), order, f, lf)
    rate = np.log2(e1 / e2)
    assert e2 < e1 and rate > order - 0.6, (e1, e2, rate)


@pytest.mark.parametrize("ckw", [dict(coord="SinhSpherical", amp=4.0, sinhw=0.6, bscale=0.0),
                                 dict(coord="SinhSymTP", amp=4.0, sinhw=0.6, bscale=1.5)])
def test_p4_harmonic_polynomial_is_annihilated(ckw):
    # x^2 - y^2 + 3 x z - 2 z has zero flat Laplacian; checks every factor's sign and the u_0/u_1 terms
    p = small(ckw, (24, 16, 16), 8)
    o = O.Oracle(p)
    xyz = grid_cart(o, p)
    x, y, z = xyz.T
    u = x**2 - y**2 + 3 * x * z - 2 * z
    lap = o.laplacian(u)[o.interior_mask()]
    lap_single_term = o.laplacian(x**2)[o.interior_mask()]  # = 2 up to truncation
    # The sinh maps stretch a polynomial in x,y,z into exponentials of x0: truncation, not
    # rounding, limits the agreement.  A dropped or mis-signed term gives O(1) here.
    assert np.median(np.abs(lap_single_term - 2.0)) < 2e-2
    assert np.median(np.abs(lap)) < 2e-2 * np.median(np.abs(lap_single_term))


# ------------------------------------------------------------------------------------------
# P5 / P7  sources: psi_BL harmonic, Bowen-York identities and closed forms (C1, C2)
# ------------------------------------------------------------------------------------------
def test_p5_psi_bl_is_harmonic_away_from_punctures():
    ckw = dict(coord="SinhSymTP", amp=6.0, sinhw=0.9, bscale=1.0)
    punct = [[0.7, 0, 0, 1.0, 0, 0, 0, 0, 0, 0], [0.4, 0, 0, -1.0, 0, 0, 0, 0, 0, 0]]
    errs = []
    for n in ((16, 16, 8), (32, 32, 16)):
        p = small(ckw, n, 4, punctures=punct)
        o = O.Oracle(p)
        psi, _ = o.source()
        xyz = grid_cart(o, p)
        far = (np.linalg.norm(xyz - [0, 0, 1.0], axis=1) > 1.5) & (np.linalg.norm(xyz + [0, 0, 1.0], axis=1) > 1.5)
        lap = o.laplacian(psi)
        sel = o.interior_mask() & far
        errs.append(np.max(np.abs(lap[sel])))
        # definition itself at a few points
        for q in (5, 1234, o.ntot - 7):
            r1, r2 = np.linalg.norm(xyz[q] - [0, 0, 1.0]), np.linalg.norm(xyz[q] + [0, 0, 1.0])
            assert psi[q] == pytest.approx(1 + 0.7 / (2 * r1) + 0.4 / (2 * r2), rel=1e-14)
    assert errs[1] < errs[0] / 8 and errs[1] < 1e-3


def test_p7_bowen_york_symmetric_tracefree_divergencefree():
    punct = [[0.8, 0, 0, 2.0, 0.08, -0.03, 0.02, 0.1, 0.05, 0.2],
             [0.2, 0.1, 0, -8.0, -0.08, 0.01, 0, 0.0, 0.03, -0.02]]
    rng = np.random.default_rng(11)
    for _ in range(20):
        x = rng.uniform(-6, 6, 3)
        A = O.bowen_york(punct, x)
        scale = np.abs(A).max()
        assert np.allclose(A, A.T, rtol=0, atol=1e-15 * scale)
        assert abs(np.trace(A)) < 1e-14 * scale
        h = 1e-3
        div = np.zeros(3)
        for j in range(3):
            e = np.zeros(3)
            e[j] = h
            # 4th-order centred difference of d_j A^{ij}
            div += (8 * (O.bowen_york(punct, x + e)[:, j] - O.bowen_york(punct, x - e)[:, j])
                    - (O.bowen_york(punct, x + 2 * e)[:, j] - O.bowen_york(punct, x - 2 * e)[:, j])) / (12 * h)
        assert np.all(np.abs(div) < 1e-8 * scale)


def test_p7_single_puncture_closed_form_contraction():
    # A_ij A^ij = 9/(2 r^4) [P^2 + 2 (P.n)^2] + 18/r^6 [S^2 - (S.n)^2] + 18/r^5 P.(S x n)
    rng = np.random.default_rng(12)
    for _ in range(20):
        P, S, pos = rng.uniform(-0.2, 0.2, 3), rng.uniform(-0.3, 0.3, 3), rng.uniform(-1, 1, 3)
        x = rng.uniform(-4, 4, 3)
        A = O.bowen_york([[1.0, *pos, *P, *S]], x)
        d = x - pos
        r = np.linalg.norm(d)
        n = d / r
        closed = (9 / (2 * r**4) * (P @ P + 2 * (P @ n) ** 2) + 18 / r**6 * (S @ S - (S @ n) ** 2)
                  + 18 / r**5 * (P @ np.cross(S, n)))
        assert np.sum(A * A) == pytest.approx(closed, rel=1e-12)


def test_p7_config0_source_closed_form_on_grid():
    # one spinning puncture at the origin: S = 18 S_z^2 sin^2(theta) / (8 r^6), psi_BL = 1 + m/(2|r|)
    p = W.config(0)
    o = O.Oracle(p)
    psi, S = o.source()
    x0, x1, x2 = o.coords()
    r = p["amp"] * np.sinh(x0 / p["sinhw"]) / np.sinh(1 / p["sinhw"])
    ref_S = 18 * 0.2**2 * np.sin(x1)[None, :, None] ** 2 / (8 * r[None, None, :] ** 6) * np.ones((o.T[2], 1, 1))
    ref_psi = 1 + 1.0 / (2 * np.abs(r))[None, None, :] * np.ones((o.T[2], o.T[1], 1))
    assert np.allclose(S.reshape(o.T[::-1]), ref_S, rtol=1e-11)
    assert np.allclose(psi.reshape(o.T[::-1]), ref_psi, rtol=1e-13)


# ------------------------------------------------------------------------------------------
# P8  wave speed and time step (C9): scale factors from a numerical Jacobian of the map
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ckw,n,order", [(SPH, (16, 8, 8), 4), (TP, (16, 12, 8), 8)])
def test_p8_cfl_identity_and_dt_bruteforce(ckw, n, order):
    p = small(ckw, n, order, cfl=0.4, c_min=1.0)
    o = O.Oracle(p)
    pl = o.planes()
    ng = order // 2
    x0, x1, _ = o.coords()
    dx = [1 / n[0], np.pi / n[1], 2 * np.pi / n[2]]
    # brute force: |d X / d x^a| dx^a by central differences of the coordinate map
    ds = np.zeros((o.T[1], o.T[0]))
    for j in range(o.T[1]):
        for i in range(o.T[0]):
            q = np.array([x0[i], x1[j], 0.37])
            vals = []
            for a in range(3):
                e = np.zeros(3)
                e[a] = 1e-6
                d = (O.map_to_cart(CID[p["coord"]], p["amp"], p["sinhw"], p["bscale"], *(q + e))
                     - O.map_to_cart(CID[p["coord"]], p["amp"], p["sinhw"], p["bscale"], *(q - e))) / 2e-6
                vals.append(np.linalg.norm(d) * dx[a])
            ds[j, i] = min(vals)
    assert np.allclose(pl["ds"], ds, rtol=1e-6)
    inner = ds[ng:-ng, ng:-ng]
    assert o.dsmin == pytest.approx(inner.min(), rel=1e-6)
    assert o.dt == pytest.approx(0.4 * o.dsmin, rel=1e-15)
    # local Courant number is CFL everywhere, c >= c_min on the interior
    assert np.allclose(pl["c"] * o.dt / pl["ds"], 0.4, rtol=1e-13)
    assert pl["c"][ng:-ng, ng:-ng].min() == pytest.approx(1.0, rel=1e-15)


# ------------------------------------------------------------------------------------------
# P9  outer radiation condition (C13): exact outgoing wave g(r - t)/r
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ckw", [dict(coord="SinhSpherical", amp=10.0, sinhw=0.6, bscale=0.0),
                                 dict(coord="SinhSymTP", amp=10.0, sinhw=0.6, bscale=3.0)])
def test_p9_outgoing_wave_is_annihilated_at_second_order(ckw):
    def G(r):
        return np.exp(-((r - 9.5) / 2.0) ** 2)

    def dG(r):
        return -2 * (r - 9.5) / 4.0 * G(r)

    errs = []
    for n in ((24, 12, 8), (48, 24, 8)):
        p = small(ckw, n, 4)
        o = O.Oracle(p)
        xyz = grid_cart(o, p)
        r = np.linalg.norm(xyz, axis=1)
        f = G(r) / r
        ku, kv = o.rhs(f, 2 * f, part="outer")
        _, _, outer = o.bc_lists()
        c = np.broadcast_to(o.planes()["c"][None], (o.T[2], o.T[1], o.T[0])).reshape(-1)
        # d_t f = -c (d_r f + f/r) = -c G'(r)/r for f = G(r - c t)/r
        exact = -c * dG(r) / r
        scale = np.max(np.abs(exact[outer]))
        errs.append(np.max(np.abs(ku[outer] - exact[outer])) / scale)
        assert np.allclose(kv[outer], 2 * ku[outer], rtol=1e-13, atol=1e-15 * scale)
        rest = np.ones(o.ntot, bool)
        rest[outer] = False
        assert not ku[rest].any() and not kv[rest].any()
    assert errs[0] < 0.3 and errs[1] < 0.08 and errs[1] < errs[0] / 3.0, errs


# ------------------------------------------------------------------------------------------
# P6 / P10 / P11 / P12 / C15  the loop
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ckw,order", [(SPH, 4), (TP, 8)])
def test_p6_vanishing_momentum_and_spin_is_an_exact_fixed_point(ckw, order):
    p = small(ckw, (12, 10, 8), order, punctures=[[0.5, 0, 0, 5.0, 0, 0, 0, 0, 0, 0],
                                                  [0.5, 0, 0, -5.0, 0, 0, 0, 0, 0, 0]])
    o = O.Oracle(p)
    _, S = o.source()
    assert not S.any()
    z = np.zeros(o.ntot)
    ku, kv = o.rhs(z, z)
    assert not ku.any() and not kv.any()
    u, v = o.step(z, z, 7)
    assert not u.any() and not v.any()
    assert o.residual(u) == 0.0


def test_p10_rk4_scalar_test_equation():
    # S = 0 and (u, v) = (const, 0): lap u = 0 (to rounding), so u' = -eta u at points whose stencils
    # never see the outer radiation layer: one step multiplies u by 1 + z + z^2/2 + z^3/6 + z^4/24
    ng = 2
    p = small(dict(coord="SinhSpherical", amp=5.0, sinhw=0.5, bscale=0.0), (40, 6, 8), 4, eta=3.0,
              punctures=[[1.0, 0, 0, 0.0, 0, 0, 0, 0, 0, 0]])
    o = O.Oracle(p)
    u0 = np.full(o.ntot, 0.75)
    u, v = o.step(u0, np.zeros(o.ntot), 1)
    z = -3.0 * o.dt
    amp = 1 + z + z**2 / 2 + z**3 / 6 + z**4 / 24
    U = u.reshape(o.T[::-1])
    V = v.reshape(o.T[::-1])
    safe = slice(ng, ng + 40 - 4 * ng * 3)  # 3 further RHS evaluations, ng points each, plus margin
    # (FD weights applied to a constant cancel only to rounding, so v is ~1e-16, not 0)
    assert np.allclose(U[ng:-ng, ng:-ng, safe], 0.75 * amp, rtol=1e-14, atol=0)
    assert np.abs(V[ng:-ng, ng:-ng, safe]).max() < 1e-12
    assert abs(z) > 1e-3  # the test is not vacuous


def test_p10_rk4_fourth_order_in_dt():
    ckw = dict(coord="SinhSpherical", amp=4.0, sinhw=0.7, bscale=0.0)
    punct = [[1.0, 0, 0, 0.0, 0, 0, 0, 0, 0, 0.3]]
    sols = []
    for cfl, steps in ((0.4, 8), (0.2, 16), (0.1, 32)):
        o = O.Oracle(small(ckw, (12, 6, 8), 4, punctures=punct, cfl=cfl, eta=1.0))
        u0, v0 = W.random_state(o.ntot, 7, amplitude=0.05)
        # smooth the seeded state along each axis so that the ODE system is not stiffness-limited
        u0 = o.apply_inner(u0)
        v0 = o.apply_inner(v0)
        u, _ = o.step(u0, v0, steps)
        sols.append(u[o.interior_mask()])
    e1, e2 = np.abs(sols[0] - sols[2]).max(), np.abs(sols[1] - sols[2]).max()
    assert np.log2(e1 / e2) > 3.6, (e1, e2)


def test_p11_config0_residual_decays_monotonically_after_transients():
    o = O.Oracle(W.config(0))
    u = np.zeros(o.ntot)
    v = np.zeros(o.ntot)
    psi, _ = o.source()
    hist = []
    for _ in range(20):
        u, v = o.step(u, v, 50)
        hist.append((o.residual(u, 0), o.residual(u, 1)))
        assert np.all(psi + u > 0)
    h = np.array(hist)
    assert np.all(np.diff(h[2:, 0]) < 0) and np.all(np.diff(h[2:, 1]) < 0)
    assert h[-1, 1] < 1e-2 * h[2, 1]


def test_p11_reduced_config1_and_config3_decay():
    for i, eta in ((1, 30.0), (3, 60.0)):
        p = W.config(i, scale=0.25 if i == 1 else 0.0625)
        p["eta"] = eta
        o = O.Oracle(p)
        u = np.zeros(o.ntot)
        v = np.zeros(o.ntot)
        hist = []
        for _ in range(16):
            u, v = o.step(u, v, 50)
            hist.append(o.residual(u, 1))
        h = np.array(hist)
        assert np.all(np.isfinite(h))
        assert np.all(np.diff(h[4:]) < 0), h
        assert h[-1] < 0.1 * h[4]


@pytest.mark.parametrize("mode", [0, 1])
def test_p12_residual_at_zero_state_is_source_only(mode):
    p = W.config(1, scale=0.25)
    o = O.Oracle(p)
    psi, S = o.source()
    norm, H = o.residual(np.zeros(o.ntot), mode, return_H=True)
    m = o.interior_mask()
    assert np.allclose(H[m], (S * psi**-7.0)[m], rtol=1e-14, atol=0)
    assert not H[~m].any()
    # weights from a numerical Jacobian (independent of the oracle's h_a formulas)
    x0, x1, _ = o.coords()
    w2d = np.zeros((o.T[1], o.T[0]))
    for j in range(o.T[1]):
        for i in range(o.T[0]):
            q = np.array([x0[i], x1[j], -1.1])
            hs = []
            for a in range(3):
                e = np.zeros(3)
                e[a] = 1e-6
                d = (O.map_to_cart(1, p["amp"], p["sinhw"], p["bscale"], *(q + e))
                     - O.map_to_cart(1, p["amp"], p["sinhw"], p["bscale"], *(q - e))) / 2e-6
                hs.append(np.linalg.norm(d))
            w2d[j, i] = np.prod(hs)
    w = np.broadcast_to(w2d[None], (o.T[2], o.T[1], o.T[0])).reshape(-1) if mode == 0 else np.ones(o.ntot)
    ref = np.sqrt(np.sum(w[m] * H[m] ** 2) / np.sum(w[m]))
    ref_rev = np.sqrt(np.sum((w[m] * H[m] ** 2)[::-1]) / np.sum(w[m][::-1]))
    assert norm == pytest.approx(ref, rel=1e-6 if mode == 0 else 1e-13)
    assert ref == pytest.approx(ref_rev, rel=1e-13)


def test_c15_inner_ghosts_stay_bitwise_equal_to_their_sources():
    p = W.config(1, scale=0.25)
    o = O.Oracle(p)
    dst, src, _ = o.bc_lists()
    u0, v0 = W.random_state(o.ntot, 21, amplitude=0.05)
    u0, v0 = o.apply_inner(u0), o.apply_inner(v0)
    u, v = o.step(u0, v0, 5)
    assert np.array_equal(u[dst], u[src]) and np.array_equal(v[dst], v[src])
    ku, kv = o.rhs(u, v)
    assert np.array_equal(ku[dst], ku[src]) and np.array_equal(kv[dst], kv[src])


def test_eq5_rhs_pointwise_from_its_parts():
    # k_u = v - eta u and k_v = c^2 (lap u + S (psi+u)^-7), assembled here from separately
    # pinned pieces (laplacian: P3/P4; source: P7; c: P8)
    p = W.config(0)
    o = O.Oracle(p)
    u, v = W.random_state(o.ntot, 1)
    ku, kv = o.rhs(u, v, part="interior")
    m = o.interior_mask()
    psi, S = o.source()
    c = np.broadcast_to(o.planes()["c"][None], (o.T[2], o.T[1], o.T[0])).reshape(-1)
    assert np.allclose(ku[m], (v - p["eta"] * u)[m], rtol=1e-15, atol=1e-17)
    ref = c**2 * (o.laplacian(u) + S * (psi + u) ** -7.0)
    assert np.allclose(kv[m], ref[m], rtol=1e-13, atol=0)
    assert not ku[~m].any() and not kv[~m].any()


def test_c19_fp32_oracle_tracks_fp64_oracle():
    p = W.config(1, scale=0.25)
    o = O.Oracle(p)
    u, v = W.random_state(o.ntot, 4)
    u, v = o.apply_inner(u), o.apply_inner(v)
    ku, kv = o.rhs(u, v)
    ku32, kv32 = o.rhs(u.astype(np.float32), v.astype(np.float32))
    assert ku32.dtype == np.float32
    assert np.abs(ku32 - ku).max() / np.abs(ku).max() < 1e-6
    assert np.abs(kv32 - kv).max() / np.abs(kv).max() < 1e-5
    r64 = o.residual(u)
    r32 = o.residual(u.astype(np.float32))
    assert r32 == pytest.approx(r64, rel=1e-4)


def test_invalid_parameters_are_rejected():
    for bad in (dict(n=(8, 6, 7)), dict(n=(1, 6, 8)), dict(fd_order=5), dict(cfl=0.0), dict(eta=-1.0),
                dict(punctures=[[0.0, 0, 0, 0, 0, 0, 0, 0, 0, 0]])):
        p = small(SPH, (8, 6, 8), 4)
        p.update(bad)
        with pytest.raises(ValueError):
            O.Oracle(p)


# ------------------------------------------------------------------------------------------
# P13  the grid-centre offset `origin` (C6): every other pin runs with origin = 0
# ------------------------------------------------------------------------------------------
def test_p13_origin_offset_enters_the_sources_with_the_right_sign_and_axis():
    """psi_BL and S on a grid whose centre is NOT the Cartesian origin equal the closed forms at
    (coordinate map + origin): a sign slip (map - origin) or an axis slip fails, because the three
    components of origin differ and the punctures sit off every axis."""
    ckw = dict(coord="SinhSymTP", amp=8.0, sinhw=0.8, bscale=2.0)
    origin = (0.3, -0.2, -3.0)
    P, S, pos, m = np.array([0.05, -0.02, 0.11]), np.array([0.1, 0.05, -0.2]), np.array([0.4, 0.7, -1.1]), 0.6
    p = small(ckw, (12, 10, 8), 4, punctures=[[m, *pos, *P, *S]], origin=origin)
    o = O.Oracle(p)
    psi, Ssrc = o.source()
    x0, x1, x2 = o.coords()
    # Cartesian position written out here (not through grid_cart / the oracle's map): C4 + C6
    A = p["amp"] * np.sinh(x0 / p["sinhw"]) / np.sinh(1 / p["sinhw"])
    X = A[None, None, :] * np.sin(x1)[None, :, None] * np.cos(x2)[:, None, None] + origin[0]
    Y = A[None, None, :] * np.sin(x1)[None, :, None] * np.sin(x2)[:, None, None] + origin[1]
    Z = np.sqrt(A**2 + p["bscale"] ** 2)[None, None, :] * np.cos(x1)[None, :, None] * np.ones_like(x2)[:, None, None] + origin[2]
    d = np.stack([X - pos[0], Y - pos[1], Z - pos[2]], axis=-1).reshape(-1, 3)
    r = np.linalg.norm(d, axis=1)
    n = d / r[:, None]
    assert np.allclose(psi, 1 + m / (2 * r), rtol=1e-13)
    closed = (9 / (2 * r**4) * (P @ P + 2 * (n @ P) ** 2) + 18 / r**6 * (S @ S - (n @ S) ** 2)
              + 18 / r**5 * (np.cross(S, n) @ P))
    assert np.allclose(Ssrc, closed / 8, rtol=1e-10)
    # and the wrong readings are far outside that tolerance (the test can tell them apart)
    for wrong in ((-0.3, 0.2, 3.0), (-3.0, -0.2, 0.3), (0.0, 0.0, 0.0)):
        dw = d - np.asarray(origin) + np.asarray(wrong)
        assert not np.allclose(psi, 1 + m / (2 * np.linalg.norm(dw, axis=1)), rtol=1e-3)


def test_p13_config3_foci_sit_on_the_punctures():
    """C6 for configs[3]: origin = (0,0,-3), b = 5 puts the SymTP foci (grid z = +-b) on the
    punctures at z = +2 and z = -8, so psi_BL peaks at the grid points next to each focus:
    smallest rho, theta next to 0 (upper focus) or pi (lower focus).  With the sign of origin
    flipped the foci would sit at z = +8 and -2 and the maxima would move."""
    p = W.config(3, scale=0.0625)
    o = O.Oracle(p)
    psi, _ = o.source()
    ng = o.ng
    P3 = psi.reshape(o.T[2], o.T[1], o.T[0])[ng:-ng, ng:-ng, ng:-ng]
    n2, n1, n0 = P3.shape
    upper, lower = P3[:, : n1 // 2, :], P3[:, n1 // 2:, :]
    ku = np.unravel_index(np.argmax(upper), upper.shape)
    kl = np.unravel_index(np.argmax(lower), lower.shape)
    assert ku[1:] == (0, 0) and kl[1:] == (n1 - n1 // 2 - 1, 0), (ku, kl)
    # the heavier puncture (m = 0.8) is the upper one, and both peaks dwarf the far field
    assert upper.max() - 1 > lower.max() - 1 > 100 * (np.median(P3) - 1)


# ------------------------------------------------------------------------------------------
# P14  the d_theta part of d_r in SinhSymTP (rad1 of C13) where it matters
# ------------------------------------------------------------------------------------------
def test_p14_symtp_radial_derivative_theta_term_at_order_one():
    """P9 again on a SymTP grid whose outer boundary lies at A ~ b, where
    d_r f = rad0 d_0 f + rad1 d_1 f has a theta part of order one (in P9 it is < 1 %).  The
    outgoing wave G(r - t)/r is still annihilated at second order, and the converged error is a
    small fraction of the theta term itself -- so dropping rad1 (error = the term) or flipping
    its sign (error = twice the term) cannot pass."""
    ckw = dict(coord="SinhSymTP", amp=3.0, sinhw=0.9, bscale=3.0)
    r0, sig = 3.4, 1.6

    def G(r):
        return np.exp(-((r - r0) / sig) ** 2)

    def dG(r):
        return -2 * (r - r0) / sig**2 * G(r)

    errs, theta_share = [], []
    for n in ((24, 16, 8), (48, 32, 8), (96, 64, 8)):
        p = small(ckw, n, 4)
        o = O.Oracle(p)
        xyz = grid_cart(o, p)
        r = np.linalg.norm(xyz, axis=1)
        f = G(r) / r
        ku, _ = o.rhs(f, f, part="outer")
        _, _, outer = o.bc_lists()
        c = np.broadcast_to(o.planes()["c"][None], (o.T[2], o.T[1], o.T[0])).reshape(-1)
        exact = -c * dG(r) / r
        scale = np.max(np.abs(exact[outer]))
        errs.append(np.max(np.abs(ku[outer] - exact[outer])) / scale)
        # analytic size of the theta term: c * rad1 * d_theta f, with r^2 = A^2 + b^2 cos^2(theta)
        # => d_theta r = -b^2 sin cos / r and rad1 = -b^2 sin cos / (r Sigma) (C13)
        x0, x1, _ = o.coords()
        A = p["amp"] * np.sinh(x0 / p["sinhw"]) / np.sinh(1 / p["sinhw"])
        b2 = p["bscale"] ** 2
        st, ct = np.sin(x1)[:, None], np.cos(x1)[:, None]
        rr = np.sqrt(A[None, :] ** 2 + b2 * ct**2)
        Sig = A[None, :] ** 2 + b2 * st**2
        dfdr = dG(rr) / rr - G(rr) / rr**2
        term = (-b2 * st * ct / (rr * Sig)) * dfdr * (-b2 * st * ct / rr)   # rad1 * d_theta f
        term = np.broadcast_to((o.planes()["c"] * term)[None], (o.T[2], o.T[1], o.T[0])).reshape(-1)
        theta_share.append(np.max(np.abs(term[outer])) / scale)
    assert theta_share[-1] > 0.05, theta_share            # the term is not negligible here
    assert errs[1] < errs[0] / 3.0 and errs[2] < errs[1] / 3.0, errs   # second order
    assert errs[2] < 0.2 * theta_share[2], (errs, theta_share)         # far below the term itself
