"""ctypes wrapper around oracle/liboracle_hr.so -- the CPU ORACLE (test infrastructure).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It never imports the CUDA package.  Argument marshalling only; every formula is
in the C files, each citing the passage of PAPER.md / reading of DESIGN.md it follows.
"""
import ctypes as C

import numpy as np

from . import build as _build

SINHSPHERICAL = 0
SINHSYMTP = 1
SINHCYLINDRICAL = 2
SINHCARTESIAN = 3

_i32p = C.POINTER(C.c_int32)
_f64p = C.POINTER(C.c_double)


class _Params(C.Structure):
    _fields_ = [
        ("n", C.c_int32 * 3),
        ("coord", C.c_int32),
        ("fd_order", C.c_int32),
        ("n_punctures", C.c_int32),
        ("amp", C.c_double),
        ("sinhw", C.c_double),
        ("bscale", C.c_double),
        ("origin", C.c_double * 3),
        ("punctures", _f64p),
        ("eta", C.c_double),
        ("cfl", C.c_double),
        ("c_min", C.c_double),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_create.restype = C.c_void_p
        _lib.orc_create.argtypes = [C.POINTER(_Params)]
        _lib.orc_destroy.argtypes = [C.c_void_p]
        _lib.orc_bc_max_frac_err.restype = C.c_double
        _lib.orc_bc_max_frac_err.argtypes = [C.c_void_p]
        _lib.orc_psi_bl.restype = C.c_double
        _lib.orc_num_threads.restype = C.c_int32
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def fd_weights(order: int):
    n = order // 2
    c1 = np.zeros(n + 1)
    d2 = np.zeros(n + 1)
    lib().orc_fd_weights(C.c_int32(order), _ptr(c1), _ptr(d2))
    return c1, d2


def map_to_cart(coord, amp, sinhw, bscale, x0, x1, x2):
    out = np.zeros(3)
    lib().orc_map_to_cart(C.c_int32(coord), C.c_double(amp), C.c_double(sinhw), C.c_double(bscale),
                          C.c_double(x0), C.c_double(x1), C.c_double(x2), _ptr(out))
    return out


def map_from_cart(coord, amp, sinhw, bscale, xyz):
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    out = np.zeros(3)
    lib().orc_map_from_cart(C.c_int32(coord), C.c_double(amp), C.c_double(sinhw),
                            C.c_double(bscale), _ptr(xyz), _ptr(out))
    return out


def metric_at(coord, amp, sinhw, bscale, x0, x1):
    h = np.zeros(3)
    g = np.zeros(5)
    lib().orc_metric_at(C.c_int32(coord), C.c_double(amp), C.c_double(sinhw), C.c_double(bscale),
                        C.c_double(x0), C.c_double(x1), _ptr(h), _ptr(g))
    return h, g


def _punct_array(punctures):
    p = np.ascontiguousarray(np.asarray(punctures, dtype=np.float64).reshape(-1, 10))
    return p


def bowen_york(punctures, xyz):
    p = _punct_array(punctures)
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    A = np.zeros(9)
    lib().orc_bowen_york(C.c_int32(p.shape[0]), _ptr(p), _ptr(xyz), _ptr(A))
    return A.reshape(3, 3)


def psi_bl(punctures, xyz):
    p = _punct_array(punctures)
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    return float(lib().orc_psi_bl(C.c_int32(p.shape[0]), _ptr(p), _ptr(xyz)))


class Oracle:
    """One grid + source set-up (fp64) with typed evolution calls.

    `params` is the neutral dict produced by hr_workloads (keys: n, coord, fd_order, amp, sinhw,
    bscale, origin, punctures [[m, x,y,z, Px,Py,Pz, Sx,Sy,Sz], ...], eta, cfl, c_min).
    """

    def __init__(self, params: dict):
        self._h = None
        L = lib()
        self._punct = _punct_array(params["punctures"])
        p = _Params()
        p.n[:] = [int(x) for x in params["n"]]
        p.coord = {"SinhSpherical": 0, "SinhSymTP": 1, "SinhCylindrical": 2, "SinhCartesian": 3}[params["coord"]]
        p.fd_order = int(params["fd_order"])
        p.n_punctures = int(self._punct.shape[0])
        p.amp = float(params["amp"])
        p.sinhw = float(params["sinhw"])
        p.bscale = float(params.get("bscale", 0.0))
        p.origin[:] = [float(x) for x in params.get("origin", (0.0, 0.0, 0.0))]
        p.punctures = self._punct.ctypes.data_as(_f64p)
        p.eta = float(params["eta"])
        p.cfl = float(params["cfl"])
        p.c_min = float(params.get("c_min", 1.0))
        h = L.orc_create(C.byref(p))
        if not h:
            raise ValueError("orc_create rejected the parameters")
        self._h = C.c_void_p(h)
        dt, dsmin = C.c_double(), C.c_double()
        ng = C.c_int32()
        T = (C.c_int32 * 3)()
        ntot, ni, no = C.c_int64(), C.c_int64(), C.c_int64()
        L.orc_info(self._h, C.byref(dt), C.byref(dsmin), C.byref(ng), T, C.byref(ntot),
                   C.byref(ni), C.byref(no))
        self.dt, self.dsmin, self.ng = dt.value, dsmin.value, ng.value
        self.T = tuple(int(t) for t in T)
        self.n = tuple(int(x) for x in params["n"])
        self.ntot, self.n_inner, self.n_outer = ntot.value, ni.value, no.value
        self.n_int = self.n[0] * self.n[1] * self.n[2]
        self.params = params

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    # ---- set-up outputs -------------------------------------------------------------------
    def coords(self):
        x = [np.zeros(t) for t in self.T]
        lib().orc_get_coords(self._h, _ptr(x[0]), _ptr(x[1]), _ptr(x[2]))
        return x

    def bc_lists(self):
        dst = np.zeros(self.n_inner, dtype=np.int32)
        src = np.zeros(self.n_inner, dtype=np.int32)
        out = np.zeros(self.n_outer, dtype=np.int32)
        lib().orc_get_bc_lists(self._h, _ptr(dst), _ptr(src), _ptr(out))
        return dst, src, out

    def bc_max_frac_err(self):
        return float(lib().orc_bc_max_frac_err(self._h))

    def source(self):
        psi = np.zeros(self.ntot)
        S = np.zeros(self.ntot)
        lib().orc_get_source(self._h, _ptr(psi), _ptr(S))
        return psi, S

    def planes(self):
        names = ["g00", "g11", "g22", "g0", "g1", "c", "w", "ds"]
        arrs = [np.zeros((self.T[1], self.T[0])) for _ in names]
        lib().orc_get_planes(self._h, *[_ptr(a) for a in arrs])
        return dict(zip(names, arrs))

    def axis2(self):
        """C25: the x2-dependent factors z22, z2, zds, zh (T2 each); 1, 0, inf, 1 for the other systems."""
        names = ["z22", "z2", "zds", "zh"]
        arrs = [np.zeros(self.T[2]) for _ in names]
        lib().orc_get_axis2(self._h, *[_ptr(a) for a in arrs])
        return dict(zip(names, arrs))

    def interior_mask(self):
        m = np.zeros((self.T[2], self.T[1], self.T[0]), dtype=bool)
        g = self.ng
        m[g:g + self.n[2], g:g + self.n[1], g:g + self.n[0]] = True
        return m.reshape(-1)

    # ---- typed evolution ------------------------------------------------------------------
    @staticmethod
    def _suf(dtype):
        dtype = np.dtype(dtype)
        if dtype == np.float64:
            return "f64"
        if dtype == np.float32:
            return "f32"
        raise TypeError(dtype)

    def _chk(self, a, dtype):
        a = np.ascontiguousarray(a, dtype=dtype)
        assert a.size == self.ntot
        return a

    def laplacian(self, u):
        u = self._chk(u, u.dtype)
        out = np.zeros_like(u)
        getattr(lib(), "orc_laplacian_" + self._suf(u.dtype))(self._h, _ptr(u), _ptr(out))
        return out

    def rhs(self, u, v, part="all"):
        """part: 'all' (a1+a2+a3), 'interior' (a1), 'outer' (a2; other entries 0)."""
        u = self._chk(u, u.dtype)
        v = self._chk(v, u.dtype)
        ku, kv = np.zeros_like(u), np.zeros_like(u)
        fn = {"all": "orc_rhs_", "interior": "orc_rhs_interior_", "outer": "orc_bc_outer_"}[part]
        getattr(lib(), fn + self._suf(u.dtype))(self._h, _ptr(u), _ptr(v), _ptr(ku), _ptr(kv))
        return ku, kv

    def apply_inner(self, f):
        f = self._chk(f, f.dtype).copy()
        getattr(lib(), "orc_bc_inner_" + self._suf(f.dtype))(self._h, _ptr(f))
        return f

    def step(self, u, v, nsteps):
        u = self._chk(u, u.dtype).copy()
        v = self._chk(v, u.dtype).copy()
        getattr(lib(), "orc_step_" + self._suf(u.dtype))(self._h, _ptr(u), _ptr(v),
                                                        C.c_int64(int(nsteps)))
        return u, v

    def residual(self, u, mode=0, return_H=False):
        u = self._chk(u, u.dtype)
        out = np.zeros(3)
        H = np.zeros_like(u) if return_H else None
        getattr(lib(), "orc_residual_" + self._suf(u.dtype))(
            self._h, _ptr(u), C.c_int32(int(mode)), _ptr(out), _ptr(H) if return_H else None)
        return (float(out[0]), H) if return_H else float(out[0])
