"""hr_residual_static (include/hr.h): the residual launch whose scratch -- work-item partials and launch counters --
sits in a static __device__ array of the library, for callers that must not allocate.  Checked against the existing
path (hr_residual_async, scratch in the solver's workspace) on two calls in a row whose inputs differ, across solvers
that share the one array (a larger plan first, so that stale partials lie behind the smaller one's), on every
reference metric and both precisions; the size limit and the variant check are exercised too.

Same kernel, same fixed reduction order (C16): the two paths agree bit for bit, which is inside every bar the other
GPU tests use (fp64 1e-10, fp32 1e-4 of the peak).  This file sorts last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import hr_workloads as W

pytestmark = pytest.mark.gpu

CASES = [
    ("config1_f64", W.config(1), "f64"),
    ("config0_f32", W.config(0), "f32"),
    ("tp_o10_ragged_f64", W.sweep_point(2, (33, 21, 12), "SinhSymTP", 10), "f64"),
    ("sph_o6_ragged_f32", W.sweep_point(0, (70, 18, 10), "SinhSpherical", 6), "f32"),
    ("cyl_o8_ragged_f64", W.sweep_point(9, (37, 22, 10), "SinhCylindrical", 8), "f64"),
    ("cart_o4_f32", W.sweep_point(11, (40, 24, 16), "SinhCartesian", 4), "f32"),
]


@pytest.fixture(scope="module")
def hr():
    import paper_2501_14030_b200 as mod
    return mod


def _pair(s, mode, static):
    import torch
    out = torch.full((2,), float("nan"), dtype=torch.float64, device=s.device)
    (s.hr_residual_static if static else s.hr_residual_async)(mode, out)
    s.synchronize()
    return out.cpu().numpy()


def test_static_scratch_residual_matches_the_workspace_path(hr):
    import torch
    solvers = []
    for k, (name, params, dtype) in enumerate(CASES):
        s = hr.Solver(dict(params, eta=0.05), dtype=dtype)
        u, v = W.random_state(s.ntot, 700 + k, amplitude=1e-3)
        s.hr_set_state(u.astype(s.npdtype), v.astype(s.npdtype))
        solvers.append((name, s))
    _pair(solvers[0][1], 0, True)  # first use on this device: module load and the address look-up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for name, s in solvers:  # one call after the other, all through the one array
        for mode in (0, 1):
            want = _pair(s, mode, False)
            got1 = _pair(s, mode, True)
            assert np.all(np.isfinite(want)) and want[0] > 0.0 and want[1] > 0.0, (name, mode, want)
            assert np.array_equal(got1, want), (name, mode, got1, want)
            s.hr_step(1)  # another input for the call that follows
            got2 = _pair(s, mode, True)
            want2 = _pair(s, mode, False)
            assert np.array_equal(got2, want2), (name, mode, got2, want2)
            assert got2[0] != got1[0], (name, mode)  # the state did move
            # hr_residual (the blocking form) sees the same numbers and no numeric flag
            norm, num, den = s.hr_residual_ex(mode)
            assert num == got2[0] and den == got2[1] and norm == np.sqrt(got2[0] / got2[1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0  # no device memory was taken by any of the calls
    for _, s in solvers:
        s.close()


def test_static_scratch_limit_and_variant_are_rejected(hr, monkeypatch):
    import torch
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    # one-plane chunks on 16 x 128 tiles x 34 planes = 69632 partial pairs > 65536
    monkeypatch.setenv("HR_TUNE_ZC", "1")
    s = hr.Solver(W.sweep_point(12, (512, 512, 34), "SinhSpherical", 4), dtype="f64")
    monkeypatch.delenv("HR_TUNE_ZC")
    with pytest.raises(hr.HrError) as e:
        s.hr_residual_static(0, out)
    assert e.value.status == 3 and "69632" in str(e.value) and "65536" in str(e.value), str(e.value)
    s.hr_residual_async(0, out)  # the workspace path serves it
    s.synchronize()
    assert np.all(np.isfinite(out.cpu().numpy()))
    s.close()
    s = hr.Solver(W.config(0), dtype="f64", variant=2)
    with pytest.raises(hr.HrError) as e:
        s.hr_residual_static(0, out)
    assert e.value.status == 1, str(e.value)
    s.close()
