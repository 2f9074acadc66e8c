"""GPU parity tests (`-m gpu`): the CUDA path, called through the C ABI (include/hr.h), against the
CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star, readings C20/C21 in DESIGN.md):
  * boundary index maps ........ bit-exact
  * one RHS evaluation ......... max_i |k_gpu - k_or| / max_i |k_or| <= 1e-12 (fp64), 1e-5 (fp32), per field,
                                 on seeded random ghost-consistent states
  * residual after N steps ..... |r_gpu - r_or| / r_or <= 1e-10 (fp64); fp32: 1e-4 of the largest
                                 residual seen so far (C21) for the state, the fp32 evaluation noise of
                                 H for the fp32 residual kernel (C21 iii); literal numbers are printed
"""
import numpy as np
import pytest

import hr_workloads as W
from oracle.hr_oracle import Oracle

pytestmark = pytest.mark.gpu

TOL_RHS = {"f64": 1e-12, "f32": 1e-5}
NP = {"f64": np.float64, "f32": np.float32}


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2501_14030_b200 as pkg
    return pkg


def consistent_state(o, seed, dtype, amplitude=0.1):
    u, v = W.random_state(o.ntot, seed, amplitude=amplitude)
    u, v = o.apply_inner(u), o.apply_inner(v)
    return u.astype(NP[dtype]), v.astype(NP[dtype])


def relmax(a, b):
    return float(np.abs(a.astype(np.float64) - b.astype(np.float64)).max() / np.abs(b).max())


SMALL = [
    ("config0", W.config(0)),
    ("config1", W.config(1)),
    ("config3_eighth", W.config(3, scale=0.125)),
    ("sph_o6_ragged", W.sweep_point(0, (70, 18, 10), "SinhSpherical", 6)),
    ("tp_o4_ragged", W.sweep_point(1, (67, 9, 6), "SinhSymTP", 4)),
    ("tp_o10_ragged", W.sweep_point(2, (33, 21, 12), "SinhSymTP", 10)),
    ("sph_o8", W.sweep_point(3, (40, 12, 16), "SinhSpherical", 8)),
    ("tp_o2", W.sweep_point(4, (20, 10, 8), "SinhSymTP", 2)),
    ("sph_o12", W.sweep_point(5, (24, 12, 12), "SinhSpherical", 12)),
    ("minimal_o10", W.sweep_point(6, (5, 5, 6), "SinhSymTP", 10)),
    # cylindrical-like reference metric (reading C24): outer points on three faces
    ("cyl_o4", W.sweep_point(8, (40, 24, 16), "SinhCylindrical", 4)),
    ("cyl_o8_ragged", W.sweep_point(9, (33, 19, 10), "SinhCylindrical", 8)),
    ("cyl_o10_ragged", W.sweep_point(10, (35, 37, 12), "SinhCylindrical", 10)),
    # Cartesian-like reference metric (reading C25): u_2 term, x2-dependent factors, six outer faces
    ("cart_o4", W.sweep_point(11, (40, 24, 16), "SinhCartesian", 4)),
    ("cart_o8_ragged", W.sweep_point(12, (33, 19, 10), "SinhCartesian", 8)),
    ("cart_o10_ragged", W.sweep_point(13, (35, 37, 12), "SinhCartesian", 10)),
]


@pytest.mark.parametrize("name,params", SMALL, ids=[n for n, _ in SMALL])
def test_boundary_maps_bit_exact(hr, name, params):
    o = Oracle(params)
    s = hr.Solver(params)
    dst, src, outer = s.hr_get_bc_lists()
    odst, osrc, oouter = o.bc_lists()
    assert np.array_equal(dst, odst) and np.array_equal(src, osrc) and np.array_equal(outer, oouter)
    assert (s.ntot, s.ng, s.T) == (o.ntot, o.ng, o.T)
    assert s.dt == pytest.approx(o.dt, rel=1e-14)
    s.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name,params", SMALL, ids=[n for n, _ in SMALL])
def test_source_terms(hr, name, params, dtype):
    o = Oracle(params)
    s = hr.Solver(params, dtype=dtype)
    psi, S = s.hr_get_source()
    opsi, oS = o.source()
    m = o.interior_mask()
    tol = 1e-12 if dtype == "f64" else 2e-7
    assert np.allclose(psi[m], opsi[m], rtol=tol, atol=0)  # psi - 1 = m/(2r): one power of r only
    # A~^ij is summed over punctures before it is squared (C2): with opposite momenta the sum
    # cancels in the far field (by ~ separation / r), so the rounding error of S scales with the
    # un-cancelled magnitude (sum_n sqrt(S_n))^2, S_n = the oracle's source of puncture n alone.
    # Conditioning (tolerance T-src): d = x_grid + origin - x_n is a difference of numbers
    # of size L_n <= r_n + 2(|x_n| + |origin|) each carrying a few ulp, so r_n = |d| has relative error
    # ~ eps L_n / r_n (large next to a SymTP focus that carries a puncture), and S_n ~ r_n^-4 ... r_n^-6
    # amplifies it 6-fold.  r_n is recovered from the oracle's single-puncture psi_BL = 1 + m/(2 r_n).
    scale = np.zeros(o.ntot)
    cond = np.ones(o.ntot)
    org = float(np.linalg.norm(params.get("origin", (0.0, 0.0, 0.0))))
    for row in params["punctures"]:
        psin, Sn = Oracle(dict(params, punctures=[row])).source()
        scale += np.sqrt(Sn)
        rn = row[0] / (2.0 * (psin - 1.0))
        Ln = rn + 2.0 * (float(np.linalg.norm(row[1:4])) + org)
        cond = np.maximum(cond, Ln / rn)
    scale = scale ** 2
    rt = 0.0 if dtype == "f64" else 1.2e-7   # fp32: fp64 value rounded once (C19)
    at = 0.0 if dtype == "f64" else 1e-37    # fp32 subnormal range
    err = np.abs(S.astype(np.float64) - oS)
    bound = (64 + 16 * cond) * 2.2e-16 * scale
    assert np.all(err[m] <= bound[m] + rt * np.abs(oS[m]) + at), \
        float((err[m] / (bound[m] + 1e-300)).max())
    s.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("name,params", SMALL, ids=[n for n, _ in SMALL])
def test_rhs_evaluation_parity(hr, name, params, dtype):
    o = Oracle(params)
    s = hr.Solver(params, dtype=dtype)
    for seed in (1, 2):
        u, v = consistent_state(o, seed, dtype)
        s.hr_set_state(u, v)
        ku, kv = s.hr_eval_rhs()
        # the arithmetic reference is the fp64 oracle on the same (rounded) inputs
        oku, okv = o.rhs(u.astype(np.float64), v.astype(np.float64))
        eu, ev = relmax(ku, oku), relmax(kv, okv)
        assert eu <= TOL_RHS[dtype] and ev <= TOL_RHS[dtype], (name, dtype, eu, ev)
        if dtype == "f32":  # and it tracks the fp32 oracle at the fp32 rounding level
            fku, fkv = o.rhs(u, v)
            assert relmax(ku, fku) <= 1e-5 and relmax(kv, fkv) <= 1e-5
        # every one of the N_tot entries is written; ghosts mirror their sources bitwise
        dst, src, _ = o.bc_lists()
        assert np.array_equal(ku[dst], ku[src]) and np.array_equal(kv[dst], kv[src])
    s.close()


@pytest.mark.parametrize("name,params", SMALL[:4], ids=[n for n, _ in SMALL[:4]])
def test_rhs_pointwise_conditioned_error(hr, name, params):
    """Stricter than the max-norm bar: at every interior point the fp64 error is small against the
    sum of the magnitudes of the terms that were added to form k_v there."""
    o = Oracle(params)
    s = hr.Solver(params)
    u, v = consistent_state(o, 3, "f64")
    s.hr_set_state(u, v)
    ku, kv = s.hr_eval_rhs()
    oku, okv = o.rhs(u, v)
    m = o.interior_mask()
    # magnitude scale of the stencil sums: c^2 * sum |g| * |u|_max / dx^2 is bounded by c^2 lap(|u|)
    # evaluated with all-positive weights; use the oracle on |u| with the sign pattern removed:
    c2 = np.broadcast_to((o.planes()["c"] ** 2)[None], (o.T[2], o.T[1], o.T[0])).reshape(-1)
    pl = o.planes()
    n = params["n"]
    dx = [1.0 / n[0], np.pi / n[1], 2 * np.pi / n[2]]
    scale2d = (np.abs(pl["g00"]) / dx[0] ** 2 + np.abs(pl["g11"]) / dx[1] ** 2 + np.abs(pl["g22"]) / dx[2] ** 2
               + np.abs(pl["g0"]) / dx[0] + np.abs(pl["g1"]) / dx[1])
    scale = c2 * np.broadcast_to(scale2d[None], (o.T[2], o.T[1], o.T[0])).reshape(-1) * 0.1 * 8.0
    err = np.abs(kv - okv)[m] / scale[m]
    assert err.max() < 1e-14, err.max()
    assert np.abs(ku - oku)[m].max() <= 4e-16 * max(1.0, params["eta"])
    s.close()


STEP_CASES = [("config0", W.config(0), 200), ("config1_half", dict(W.config(1, scale=0.5), eta=30.0), 400),
              ("config3_eighth", dict(W.config(3, scale=0.125), eta=60.0), 200),
              ("sph_o6_ragged", dict(W.sweep_point(0, (70, 18, 10), "SinhSpherical", 6), eta=2.0), 100),
              # (eta dt must stay well below RK4's real-axis limit 2.78, C10: dt = 3.2 and 1.7 on these coarse grids)
              ("cyl_o8_ragged", dict(W.sweep_point(9, (33, 38, 10), "SinhCylindrical", 8), eta=0.2), 100),
              ("cyl_o4", dict(W.sweep_point(8, (40, 48, 16), "SinhCylindrical", 4), eta=0.2), 200),
              ("cart_o8_ragged", dict(W.sweep_point(12, (33, 38, 26), "SinhCartesian", 8), eta=0.02), 100),
              ("cart_o4", dict(W.sweep_point(11, (40, 48, 32), "SinhCartesian", 4), eta=0.02), 200)]


@pytest.mark.parametrize("name,params,steps", STEP_CASES, ids=[c[0] for c in STEP_CASES])
def test_residual_after_n_steps_fp64(hr, name, params, steps):
    o = Oracle(params)
    s = hr.Solver(params)
    z = np.zeros(o.ntot)
    ou, ov = z.copy(), z.copy()
    done = 0
    for mark in (steps // 4, steps):
        s.hr_step(mark - done)
        ou, ov = o.step(ou, ov, mark - done)
        done = mark
        for mode in (0, 1):
            r, ro = s.hr_residual(mode), o.residual(ou, mode)
            assert abs(r - ro) <= 1e-10 * ro, (name, mark, mode, r, ro)
    u, v = s.hr_get_u(), s.hr_get_v()
    assert relmax(u, ou) <= 1e-11 and relmax(v, ov) <= 1e-9
    dst, src, _ = o.bc_lists()
    assert np.array_equal(u[dst], u[src]) and np.array_equal(v[dst], v[src])
    s.close()


def test_config1_full_2000_steps_fp64(hr):
    params = W.config(1)
    o = Oracle(params)
    s = hr.Solver(params)
    z = np.zeros(o.ntot)
    s.hr_step(params["steps"])
    ou, ov = o.step(z, z, params["steps"])
    for mode in (0, 1):
        r, ro = s.hr_residual(mode), o.residual(ou, mode)
        # C21(ii): after 2000 steps the residual has fallen ~7 decades below its start value, H is the
        # rounding-level remainder of two cancelling terms, and the attainable agreement is 1e-10 of the
        # LARGEST residual of the run (the one at u = 0), not of the current one; the literal relative
        # number is printed and held to a looser sanity bound.
        peak = max(ro, o.residual(z, mode))
        print(f"config1 mode {mode}: gpu {r:.15e} oracle {ro:.15e} literal rel {abs(r - ro) / ro:.2e} "
              f"decay {ro / peak:.1e}")
        assert abs(r - ro) <= 1e-10 * peak, (mode, r, ro, peak)
        assert abs(r - ro) <= 1e-5 * ro, (mode, r, ro)
    assert relmax(s.hr_get_u(), ou) <= 1e-10
    s.close()


def test_fp32_residual_history_against_fp64_oracle(hr):
    """configs[2]'s comparison on a reduced grid: fp32 GPU vs fp64 oracle, every 100 steps."""
    params = dict(W.config(2, scale=0.25), eta=60.0)
    o = Oracle(params)
    s32 = hr.Solver(params, dtype="f32", residual_mode=1)
    s64 = hr.Solver(params, dtype="f64", residual_mode=1)
    z = np.zeros(o.ntot)
    ou, ov = z.copy(), z.copy()
    ou32, ov32 = z.astype(np.float32), z.astype(np.float32)
    peak = o.residual(z, 1)  # C21: the scale is max over n <= N of r_or64(n), n = 0 (u = 0) included
    e_or = floor = miss = 0.0
    bad = []
    print(f"peak (n = 0) {peak:.6e}")
    for it in range(6):
        s32.hr_step(100)
        s64.hr_step(100)
        ou, ov = o.step(ou, ov, 100)
        ou32, ov32 = o.step(ou32, ov32, 100)
        ro = o.residual(ou, 1)
        peak = max(peak, ro)
        r32, r64 = s32.hr_residual(), s64.hr_residual()
        print(f"step {100 * (it + 1)}: oracle64 {ro:.6e} gpu64 rel {abs(r64 - ro) / ro:.2e} "
              f"gpu32 rel {abs(r32 - ro) / ro:.2e} oracle32 rel {abs(o.residual(ou32, 1) - ro) / ro:.2e}")
        assert abs(r64 - ro) <= 1e-10 * ro
        # FROZEN BARS (they change only in a commit that touches no kernel):
        # (a) SURVEY C21: |r_gpu32 - r_or64| <= 1e-4 * max_{n <= N} r_or64(n), the literal number printed above.
        # Two fp32 roundings of one run are two noise samples, so the comparison is between envelopes: the
        # GPU's largest miss over the run <= max(1e-4 * peak, 1.5 x the fp32 ORACLE's largest miss over the
        # run) -- asserted after the loop (tests/test_gpu_full_configs.py applies the same rule at full size,
        # and the plain 1e-4 * peak on configs[2] itself).
        floor = max(floor, abs(o.residual(ou32, 1) - ro))
        miss = max(miss, abs(r32 - ro))
        # (b) C21 (iii), GPU-vs-fp32-oracle drift: the GPU's fp32 state may not sit further from the fp64
        # oracle's than 1.5x what the fp32 ORACLE's state does (plus 4 ulp32 of max|u|), and the residual
        # of that state, evaluated in fp64 by the oracle, within 1e-4 * peak + 1.5x the largest miss the
        # fp32 oracle's own state has shown so far (two fp32 roundings of one run are two noise samples).
        u32 = s32.hr_get_u()
        eg = np.abs(u32.astype(np.float64) - ou).max()
        eo = np.abs(ou32.astype(np.float64) - ou).max()
        r_state64 = o.residual(u32.astype(np.float64), 1)
        r_state32 = o.residual(u32, 1)
        e_or = max(e_or, abs(o.residual(ou32.astype(np.float64), 1) - ro))
        # (c) the GPU's fp32 residual KERNEL against the fp32 oracle's residual of the same state: within
        # the evaluation noise of H in fp32, measured as fp32 vs fp64 oracle evaluation of fp32 states
        noise = max(abs(r_state32 - r_state64), abs(o.residual(ou32, 1) - o.residual(ou32.astype(np.float64), 1)))
        print(f"          fp32 state vs fp64 oracle: gpu {eg / np.abs(ou).max():.2e} fp32 oracle {eo / np.abs(ou).max():.2e} "
              f"(of max|u|); its residual in fp64: rel {abs(r_state64 - ro) / ro:.2e} (fp32 oracle so far: "
              f"{e_or / ro:.2e}); evaluation noise {noise / ro:.2e}; gpu32 vs oracle32 on that state "
              f"{abs(r32 - r_state32) / ro:.2e}")
        if eg > 1.5 * eo + 4 * np.finfo(np.float32).eps * np.abs(ou).max():
            bad.append(("b-state", it, eg, eo))
        if abs(r_state64 - ro) > 1e-4 * peak + 1.5 * e_or:
            bad.append(("b-residual", it, r_state64, ro, e_or))
        if abs(r32 - r_state32) > 1e-4 * peak + 2.0 * noise:
            bad.append(("c", it, r32, r_state32, noise))
    print(f"largest miss over the run: gpu32 {miss / peak:.2e} fp32 oracle {floor / peak:.2e} (of peak)")
    assert miss <= max(1e-4 * peak, 1.5 * floor), (miss, floor, peak)
    assert not bad, bad
    s32.close()
    s64.close()


def test_fixed_point_zero_momentum_zero_spin(hr):
    params = dict(W.config(1, scale=0.25))
    params["punctures"] = [[0.5, 0, 0, 5.0, 0, 0, 0, 0, 0, 0], [0.5, 0, 0, -5.0, 0, 0, 0, 0, 0, 0]]
    for dtype in ("f64", "f32"):
        s = hr.Solver(params, dtype=dtype)
        _, S = s.hr_get_source()
        assert not S.any()
        s.hr_step(5)
        assert not s.hr_get_u().any() and not s.hr_get_v().any()
        assert s.hr_residual() == 0.0
        s.close()


def test_no_punctures_and_set_state_fills_ghosts(hr):
    params = dict(W.config(0), punctures=[])
    o = Oracle(params)
    s = hr.Solver(params)
    u, v = W.random_state(o.ntot, 9)  # NOT ghost-consistent
    s.hr_set_state(u, v)
    got = s.hr_get_u()
    assert np.array_equal(got, o.apply_inner(u))
    s.close()


def test_full_size_config3_rhs_and_two_steps(hr):
    """BASELINE configs[3] at its full size (512x256x64, 10th order): one RHS evaluation over all
    10 275 048 points and the residual after 2 RK4 steps, in the launch configuration bench.py times."""
    params = W.config(3)
    o = Oracle(params)
    s = hr.Solver(params)
    dst, src, outer = s.hr_get_bc_lists()
    odst, osrc, oouter = o.bc_lists()
    assert np.array_equal(dst, odst) and np.array_equal(src, osrc) and np.array_equal(outer, oouter)
    u, v = consistent_state(o, 5, "f64")
    s.hr_set_state(u, v)
    ku, kv = s.hr_eval_rhs()
    oku, okv = o.rhs(u, v)
    assert relmax(ku, oku) <= 1e-12 and relmax(kv, okv) <= 1e-12
    z = np.zeros(o.ntot)
    s.hr_set_state(z, z)
    s.hr_step(2)
    ou, ov = o.step(z, z, 2)
    r, ro = s.hr_residual(1), o.residual(ou, 1)
    assert abs(r - ro) <= 1e-10 * ro
    assert relmax(s.hr_get_u(), ou) <= 1e-12
    s.close()


def test_full_size_config2_fp32_rhs(hr):
    params = W.config(2)
    o = Oracle(params)
    s = hr.Solver(params, dtype="f32")
    u, v = consistent_state(o, 6, "f32")
    s.hr_set_state(u, v)
    ku, kv = s.hr_eval_rhs()
    oku, okv = o.rhs(u.astype(np.float64), v.astype(np.float64))
    assert relmax(ku, oku) <= 1e-5 and relmax(kv, okv) <= 1e-5
    s.close()


def test_largest_sweep_point_sampled(hr):
    """configs[4]'s largest grid (512x256x256, 10th order, fp32): too big to step on the oracle in
    seconds, so compare one RHS evaluation on a sampled set of i2-planes via properties that hold at
    any size: the oracle's interior formula is local, so planes can be checked one sub-grid at a time."""
    params = W.sweep_point(23, (512, 256, 256), "SinhSymTP", 10)
    s = hr.Solver(params, dtype="f32")
    ntot = s.ntot
    u, v = W.random_state(ntot, 77, dtype=np.float32)
    s.hr_set_state(u, v)
    ku, kv = s.hr_eval_rhs()
    got_u = s.hr_get_u()
    dst, src, outer = s.hr_get_bc_lists()
    # properties: ghost consistency of state and k; k_u = v - eta u on the interior
    assert np.array_equal(got_u[dst], got_u[src])
    assert np.array_equal(ku[dst], ku[src]) and np.array_equal(kv[dst], kv[src])
    T = s.T
    ng = s.ng
    U = got_u.reshape(T[2], T[1], T[0])
    V = s.hr_get_v().reshape(T[2], T[1], T[0])
    KU = ku.reshape(T[2], T[1], T[0])
    inner = (slice(ng, -ng), slice(ng, -ng), slice(ng, -ng))
    ref = V[inner] - np.float32(params["eta"]) * U[inner]
    assert np.allclose(KU[inner], ref, rtol=1e-6, atol=1e-6)
    # sampled oracle comparison of k_v: a thin slab in i2 has the same interior arithmetic because no
    # factor depends on x2 except through u, psi, S (C4); build a slab oracle with the same punctures
    # rotated?  phi enters psi and S, so instead compare against the full-size oracle's interior RHS.
    o = Oracle(params)
    oku, okv = o.rhs(got_u.astype(np.float64), V.reshape(-1).astype(np.float64), part="interior")
    m = o.interior_mask()
    assert relmax(kv[m], okv[m]) <= 1e-5 and relmax(ku[m], oku[m]) <= 1e-5
    s.close()


@pytest.mark.parametrize("variant", [1, 2, 3], ids=["paper_arrangement", "direct_fused", "running_sum_rk4"])
@pytest.mark.parametrize("name,params", [SMALL[0], SMALL[3], SMALL[5]], ids=[SMALL[0][0], SMALL[3][0], SMALL[5][0]])
def test_other_arrangements_match_oracle(hr, name, params, variant):
    """The other arrangements (variant 1: the paper's RHS -> BC -> RK kernels with k in HBM, SURVEY.md f4;
    variant 2: round-1a direct-load fused kernel; variant 3: the marching kernels with RK4 as a running
    sum, the default's predecessor) meet the same bars as the default."""
    o = Oracle(params)
    for dtype in ("f64", "f32"):
        s = hr.Solver(params, dtype=dtype, variant=variant)
        u0, v0 = consistent_state(o, 5, dtype)
        s.hr_set_state(u0, v0)
        ku, kv = s.hr_eval_rhs()
        oku, okv = o.rhs(u0.astype(np.float64), v0.astype(np.float64))
        assert relmax(ku, oku) <= TOL_RHS[dtype] and relmax(kv, okv) <= TOL_RHS[dtype]
        s.close()
    s = hr.Solver(params, variant=variant)
    z = np.zeros(o.ntot)
    s.hr_step(20)
    ou, ov = o.step(z, z, 20)
    for mode in (0, 1):
        r, ro = s.hr_residual(mode), o.residual(ou, mode)
        assert abs(r - ro) <= 1e-10 * ro, (mode, r, ro)
    u = s.hr_get_u()
    dst, src, _ = o.bc_lists()
    assert np.array_equal(u[dst], u[src])
    s.close()


def test_relaxation_loop_with_stopping_criterion(hr):
    """hr_relax (Alg. 1 l.8-18): residual history equals the oracle's, block by block, and the loop stops
    one block after the first residual <= tol (the host tests a residual while the next block runs)."""
    params = W.config(0)
    o = Oracle(params)
    every = 20
    z = np.zeros(o.ntot)
    ou, ov = z.copy(), z.copy()
    ref = [o.residual(ou, 0)]
    for _ in range(10):
        ou, ov = o.step(ou, ov, every)
        ref.append(o.residual(ou, 0))
    ref = np.array(ref)
    assert np.all(np.diff(ref[3:]) < 0)  # decaying after the transient (P11), so a threshold is meaningful
    j = 6
    tol = float(np.sqrt(ref[j] * ref[j - 1]))  # between two checks: the decision is not borderline
    s = hr.Solver(params)
    done, res, hist = s.hr_relax(10_000, every, tol, 0)
    assert done == (j + 1) * every, (done, j)
    assert len(hist) == j + 2
    assert np.all(np.abs(hist - ref[:j + 2]) <= 1e-10 * ref[:j + 2])
    assert res == hist[-1]
    # tol = 0 runs max_steps (ragged last block)
    s2 = hr.Solver(params)
    done2, res2, hist2 = s2.hr_relax(50, every, 0.0, 0)
    assert done2 == 50 and len(hist2) == 4
    s3 = hr.Solver(params)
    s3.hr_step(50)
    assert res2 == s3.hr_residual(0)
    for x in (s, s2, s3):
        x.close()


def test_batched_independent_grids(hr):
    """hr_step_many: N independent solvers advanced together on their own streams give,
    bit for bit, what each gives alone; one of them is checked against the oracle."""
    ps = [W.sweep_point(40 + i, (32, 16, 8), "SinhSymTP", 6) for i in range(3)]
    ps.append(W.config(0))
    together = [hr.Solver(p) for p in ps]
    hr.hr_step_many(together, 15)
    for p, s in zip(ps, together):
        alone = hr.Solver(p)
        alone.hr_step(15)
        assert np.array_equal(s.hr_get_u(), alone.hr_get_u()) and np.array_equal(s.hr_get_v(), alone.hr_get_v())
        alone.close()
    o = Oracle(ps[0])
    z = np.zeros(o.ntot)
    ou, _ = o.step(z, z, 15)
    r, ro = together[0].hr_residual(0), o.residual(ou, 0)
    assert abs(r - ro) <= 1e-10 * ro
    for s in together:
        s.close()


@pytest.mark.parametrize("name,params", [SMALL[0], SMALL[4], SMALL[5], SMALL[9]],
                         ids=[SMALL[0][0], SMALL[4][0], SMALL[5][0], SMALL[9][0]])
def test_step_with_fused_residual(hr, name, params):
    """hr_step_residual_async: the residual reduced by the first RK substep equals hr_residual of the
    state before the step (same formula and summation order; the two kernel instantiations may contract
    FMAs differently, so equal to a few ulp, not bitwise), and the step is bit for bit the same step."""
    import torch
    o = Oracle(params)
    for dtype in ("f64", "f32"):
        a = hr.Solver(params, dtype=dtype)
        b = hr.Solver(params, dtype=dtype)
        # amplitude 1e-3: a step from white noise of amplitude 0.1 drives psi_BL + u through zero on the
        # 5-point grid (|v| reaches 1e12), which the library now reports as HR_ERR_NUMERIC
        u0, v0 = consistent_state(o, 11, dtype, amplitude=1e-3)
        a.hr_set_state(u0, v0)
        b.hr_set_state(u0, v0)
        for mode in (0, 1):
            out2 = torch.zeros(2, dtype=torch.float64, device=a.device)
            ref3 = b.hr_residual_ex(mode)
            a.hr_step_residual_async(mode, out2)
            b.hr_step(1)
            a.synchronize()
            num, den = (float(x) for x in out2.cpu())
            tol = 1e-13 if dtype == "f64" else 1e-6
            assert abs(num - ref3[1]) <= tol * ref3[1] and den == ref3[2], (dtype, mode, num, ref3)
            assert np.array_equal(a.hr_get_u(), b.hr_get_u()) and np.array_equal(a.hr_get_v(), b.hr_get_v())
        a.close()
        b.close()


def test_work_item_order_knobs_do_not_change_results(hr, monkeypatch):
    """The work-item decode of the marching kernels (long items = segments of chunks, then single chunks, ragged
    last chunk and last segment): tuning knobs HR_TUNE_COL / HR_TUNE_ZC change the order in which work runs and
    how it is cut, never what is computed.  The grid has more tiles than CTA slots so that long items occur."""
    params = W.sweep_point(7, (70, 1200, 14), "SinhSymTP", 6)
    o = Oracle(params)
    for dtype in ("f64", "f32"):
        u0, v0 = consistent_state(o, 21, dtype)
        ref = None
        for gt, zc in ((None, None), ("7", "3"), ("10", "5"), ("1", "14"), ("0", "2")):
            if gt is None:
                monkeypatch.delenv("HR_TUNE_COL", raising=False)
                monkeypatch.delenv("HR_TUNE_ZC", raising=False)
            else:  # gt: here "long items on / off" (HR_TUNE_COL; 0 = single chunks only)
                monkeypatch.setenv("HR_TUNE_COL", "0" if gt == "0" else "1")
                monkeypatch.setenv("HR_TUNE_ZC", zc)
            s = hr.Solver(params, dtype=dtype)
            s.hr_set_state(u0, v0)
            ku, kv = s.hr_eval_rhs()
            s.hr_step(3)
            got = (ku, kv, s.hr_get_u(), s.hr_get_v())
            s.close()
            if ref is None:
                ref = got
                oku, okv = o.rhs(u0.astype(np.float64), v0.astype(np.float64))
                assert relmax(ku, oku) <= TOL_RHS[dtype] and relmax(kv, okv) <= TOL_RHS[dtype]
            else:
                for a, b in zip(got, ref):
                    assert np.array_equal(a, b)


def test_programmatic_launch_trigger_placement_changes_nothing(hr, monkeypatch):
    """HR_TUNE_PDL moves griddepcontrol.launch_dependents (never early / early where every CTA has one item / always at
    entry): the next substep may only START earlier, it reads nothing before its predecessor has completed, so the
    state after some steps and the fused residual are bit for bit the same -- on a grid with one item per CTA
    (config 0), one with items handed out dynamically (70 x 1200 x 14, long items) and through hr_step_many."""
    import torch
    for params in (W.config(0), W.sweep_point(7, (70, 1200, 14), "SinhSymTP", 6)):
        for dtype in ("f64", "f32"):
            ref = None
            for pdl in (None, "0", "1", "2"):
                if pdl is None:
                    monkeypatch.delenv("HR_TUNE_PDL", raising=False)
                else:
                    monkeypatch.setenv("HR_TUNE_PDL", pdl)
                s, t = hr.Solver(params, dtype=dtype), hr.Solver(params, dtype=dtype)
                out = torch.zeros(2, dtype=torch.float64, device="cuda")
                for _ in range(6):
                    s.hr_step_residual_async(0, out)
                s.hr_step(5)
                hr.hr_step_many([t], 11)
                s.synchronize()
                got = (s.hr_get_u(), s.hr_get_v(), out.cpu().numpy(), t.hr_get_u())
                s.close()
                t.close()
                assert np.array_equal(got[0], got[3])
                if ref is None:
                    ref = got
                    assert np.all(np.isfinite(got[2])) and got[2][0] > 0.0
                else:
                    for a, b in zip(got, ref):
                        assert np.array_equal(a, b), (params["n"], dtype, pdl)
    monkeypatch.delenv("HR_TUNE_PDL", raising=False)


@pytest.mark.parametrize("name,params", [SMALL[0], SMALL[5], SMALL[4], SMALL[3]],
                         ids=[SMALL[0][0], SMALL[5][0], SMALL[4][0], SMALL[3][0]])
def test_poisoned_workspace_changes_nothing(hr, name, params):
    """compute-sanitizer is closed on this GPU pool (profiles/r2_sanitizer.md), so initcheck's question is asked
    directly: with every byte of the caller's workspace set to 0xFF (NaN in both precisions) before hr_create,
    every result -- k, the state after steps, both residual modes, the relaxation history -- is bit for bit
    what an all-zero workspace gives, i.e. the library reads no byte it has not written (row pads of the
    stored layout and the stage buffers included)."""
    import torch
    o = Oracle(params)
    for dtype in ("f64", "f32"):
        got = []
        for poison in (False, True):
            s = hr.Solver(params, dtype=dtype, poison=poison)
            u0, v0 = consistent_state(o, 4, dtype, amplitude=1e-3)
            s.hr_set_state(u0, v0)
            ku, kv = s.hr_eval_rhs()
            z = np.zeros(o.ntot, dtype=NP[dtype])
            s.hr_set_state(z, z)
            s.hr_step(2)
            out2 = torch.zeros(2, dtype=torch.float64, device=s.device)
            s.hr_step_residual_async(1, out2)
            s.synchronize()
            done, res, hist = s.hr_relax(3, 2, 0.0, 0)
            got.append((ku, kv, s.hr_get_u(), s.hr_get_v(), out2.cpu().numpy(), np.asarray(hist),
                        np.array([s.hr_residual(0), s.hr_residual(1)])))
            assert s.hr_query("numeric_flag") == 0
            s.close()
        for a, b in zip(*got):
            assert np.array_equal(a, b) and np.isfinite(a).all()


def test_query_and_measurement_hooks(hr):
    """hr_query (which path runs, the plan, the numeric flag) and the two measurement hooks of include/hr.h."""
    s = hr.Solver(W.config(1))
    assert s.hr_query("step_graph") == 1          # hr_step replays the captured graph, not the fallback
    assert s.hr_query("persistent") == 0
    assert s.hr_query("numeric_flag") == 0
    zc, items, grid = s.hr_query("plan_zc"), s.hr_query("plan_items"), s.hr_query("plan_grid")
    assert 1 <= zc <= 16 and items >= 64 and 1 <= grid <= items
    import torch
    out2 = torch.zeros(2, dtype=torch.float64, device=s.device)
    s.hr_step_residual_async(0, out2)
    s.synchronize()
    assert s.hr_query("resid_graph") & 1
    # a state that drives psi_BL + u through zero is reported, and a new state clears the flag
    bad = np.full(s.ntot, -5.0)
    s.hr_set_state(bad, np.zeros(s.ntot))
    with pytest.raises(hr.HrError) as e:
        s.hr_residual(0)
    assert e.value.status == 5 and s.hr_query("numeric_flag") != 0
    s.hr_set_state(np.zeros(s.ntot), np.zeros(s.ntot))
    assert s.hr_query("numeric_flag") == 0 and s.hr_residual(0) > 0
    s.close()
    f64, f32 = hr.hr_measure_alu_peak("f64"), hr.hr_measure_alu_peak("f32", packed=True)
    assert 15.0 < f64 < 60.0 and 40.0 < f32 < 120.0 and f32 > 1.5 * f64, (f64, f32)  # TFLOP/s on a B200
    floor = hr.hr_measure_launch_floor(4, 148, 128, 200)
    assert 1.0 < floor < 50.0, floor  # microseconds per replay of a 4-launch graph


def _random_case(seed):
    rng = np.random.default_rng(9000 + seed)
    order = int(rng.choice([2, 4, 6, 8, 10, 12]))
    ng = order // 2
    coord = ["SinhSpherical", "SinhSymTP", "SinhCylindrical", "SinhCartesian"][seed % 4]
    n = (int(rng.integers(ng, 81)), int(rng.integers(ng, 41)), 2 * int(rng.integers((max(ng, 2) + 1) // 2, 13)))
    return dict(W.sweep_point(300 + seed, n, coord, order), eta=0.05)


@pytest.mark.parametrize("seed", range(32))
def test_random_small_grids(hr, seed):
    """Seeded random shapes (N_a from NG up, odd sizes, fewer points than a tile, every FD order, all four reference
    metrics, both precisions): boundary lists bit-exact, one RHS evaluation at the north_star bars on every one of
    the N_tot entries, ghosts bitwise equal to their sources."""
    params = _random_case(seed)
    o = Oracle(params)
    for dtype in ("f64", "f32"):
        s = hr.Solver(params, dtype=dtype)
        for a, b in zip(s.hr_get_bc_lists(), o.bc_lists()):
            assert np.array_equal(a, b), (params["coord"], params["n"], params["fd_order"])
        u, v = consistent_state(o, 50 + seed, dtype)
        s.hr_set_state(u, v)
        ku, kv = s.hr_eval_rhs()
        oku, okv = o.rhs(u.astype(np.float64), v.astype(np.float64))
        eu, ev = relmax(ku, oku), relmax(kv, okv)
        assert eu <= TOL_RHS[dtype] and ev <= TOL_RHS[dtype], (params["coord"], params["n"], params["fd_order"], dtype, eu, ev)
        dst, src, _ = o.bc_lists()
        assert np.array_equal(ku[dst], ku[src]) and np.array_equal(kv[dst], kv[src])
        s.close()
