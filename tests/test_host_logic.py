"""CPU tests (`-m "not gpu"`) of the CUDA library's HOST logic through the C ABI: the library
loads, exports every symbol include/hr.h declares, validates arguments, and its host-side set-up
(closed-form integer boundary maps, dt, coefficient planes) agrees with the oracle -- the maps
bit-exactly.  No compute call is made (there is no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import hr_workloads as W
from oracle.hr_oracle import Oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hr():
    from paper_2501_14030_b200 import build
    build.build()
    import paper_2501_14030_b200 as pkg
    return pkg


def test_library_exports_every_declared_symbol(hr):
    text = open(os.path.join(ROOT, "include", "hr.h")).read()
    names = re.findall(r"HR_API\s+[\w\s\*]+?\b(hr_\w+)\s*\(", text)
    assert len(names) >= 18 and "hr_create" in names and "hr_step" in names
    for n in names:
        assert hasattr(hr.lib, n), n
    assert "sm_100a" in hr.hr_version()


def test_struct_layout_matches_header(hr):
    # hr_puncture = 10 packed doubles; hr_params field order as in include/hr.h
    assert C.sizeof(hr.hr_puncture) == 80
    text = open(os.path.join(ROOT, "include", "hr.h")).read()
    body = text[text.index("typedef struct {\n  int32_t n[3];"):text.index("} hr_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = re.findall(r"^\s*(?:const\s+)?[\w\*]+\*?\s+([\w, \*\[\]0-9]+);", body, flags=re.M)
    flat = []
    for f in fields:
        for name in f.split(","):
            flat.append(re.sub(r"[\*\[\]0-9 ]", "", name))
    assert flat == [n for n, _ in hr.hr_params._fields_]


def test_argument_validation(hr):
    good = W.config(0)
    p, keep = hr.make_params(good)
    assert hr.hr_workspace_bytes(p) > 10 * 27200 * 8
    for bad, status in ((dict(n=(64, 16, 15)), 1), (dict(n=(1, 16, 16)), 1), (dict(fd_order=5), 2),
                        (dict(cfl=0.0), 1), (dict(eta=-1.0), 1), (dict(fd_order=14), 2)):
        q = dict(good)
        q.update(bad)
        p, keep = hr.make_params(q)
        with pytest.raises(hr.HrError) as e:
            hr.hr_workspace_bytes(p)
        assert e.value.status == status
    q = dict(good, punctures=[[0.0, 0, 0, 0, 0, 0, 0, 0, 0, 0]])
    p, keep = hr.make_params(q)
    with pytest.raises(hr.HrError):
        hr.hr_workspace_bytes(p)
    # NULL handles
    assert hr.lib.hr_step(None, 1) == 1
    assert hr.lib.hr_destroy(None) == 0
    assert b"NULL" in hr.lib.hr_last_error()


CASES = [W.config(0), W.config(1), W.config(1, scale=0.3), W.config(3, scale=0.1),
         W.sweep_point(0, (12, 10, 8), "SinhSpherical", 6),
         W.sweep_point(1, (12, 10, 8), "SinhSymTP", 12),
         W.sweep_point(2, (7, 5, 6), "SinhSpherical", 10),
         W.sweep_point(3, (16, 4, 4), "SinhSymTP", 2),
         W.sweep_point(4, (12, 10, 8), "SinhCylindrical", 4),   # reading C24
         W.sweep_point(5, (9, 7, 6), "SinhCylindrical", 10),
         W.sweep_point(6, (10, 12, 8), "SinhCartesian", 4),     # reading C25
         W.sweep_point(7, (7, 9, 12), "SinhCartesian", 8)]


@pytest.mark.parametrize("params", CASES, ids=lambda p: f"{p['name']}-{p['coord']}-o{p['fd_order']}")
def test_host_setup_matches_oracle(hr, params):
    o = Oracle(params)
    h = hr.hr_host_setup(params)
    dst, src, outer = o.bc_lists()
    # integer work: bit-exact (closed form in the library vs fp64 round trip in the oracle)
    assert np.array_equal(h["inner_dst"], dst)
    assert np.array_equal(h["inner_src"], src)
    assert np.array_equal(h["outer_idx"], outer)
    assert h["dt"] == pytest.approx(o.dt, rel=1e-14)
    assert h["dsmin"] == pytest.approx(o.dsmin, rel=1e-14)
    # coefficient planes: the library folds 1/dx^a into them
    pl = o.planes()
    n = params["n"]
    dx = [1.0 / n[0], (2.0 if params["coord"] == "SinhCylindrical" else np.pi) / n[1], 2 * np.pi / n[2]]
    if params["coord"] == "SinhCartesian":
        dx = [2.0 / n[0], 2.0 / n[1], 2.0 / n[2]]
    ng = o.ng
    inner = (slice(ng, -ng), slice(ng, -ng))  # factors are only used at interior (i0,i1)
    for name, ref in (("L00", pl["g00"] / dx[0] ** 2), ("L11", pl["g11"] / dx[1] ** 2),
                      ("L22", pl["g22"] / dx[2] ** 2), ("L0", pl["g0"] / dx[0]),
                      ("L1", pl["g1"] / dx[1]), ("W", pl["w"])):
        atol = 0.0
        if name == "L0" and params["coord"] == "SinhCylindrical":
            # C24: g0 = 1/(R R') - R''/R'^3 cancels to ~ e^(-2 x0/W) of its terms at large x0 (sinh ~ cosh), so two
            # correct evaluations differ by rounding relative to the TERMS, 1/(R R') = sqrt(g00 g22)
            assert np.all(np.abs(h["planes"][name] - ref)[inner] <= 1e-12 * np.abs(ref[inner])
                          + 8e-16 * (np.sqrt(pl["g00"] * pl["g22"]) / dx[0])[inner]), name
            continue
        assert np.allclose(h["planes"][name][inner], ref[inner], rtol=1e-12, atol=atol), name
    # c^2 is needed at interior and outer columns
    assert np.allclose(h["planes"]["C2"][ng:-ng, ng:], pl["c"][ng:-ng, ng:] ** 2, rtol=1e-13)
