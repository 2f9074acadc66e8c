"""Thin Python binding of include/hr.h (same names, argument marshalling only).

PyTorch is used for device memory (the workspace tensor, output tensors) and the CUDA stream;
every step of the hot path runs in the kernels of libhr_b200.so.  There is no CPU fallback: if
the library is missing, importing this module raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# HR_B200_LIB=libhr_b200_nofmad.so selects the --fmad=false twin of the library (same sources, the ablation of
# PAPER.md:193, 301-321; built by build.py next to the product library); a file name inside this directory only
LIB_PATH = os.path.join(_HERE, os.path.basename(os.environ.get("HR_B200_LIB", "libhr_b200.so")))

HR_OK = 0
HR_SINHSPHERICAL, HR_SINHSYMTP, HR_SINHCYLINDRICAL, HR_SINHCARTESIAN = 0, 1, 2, 3
HR_F64, HR_F32 = 0, 1
_STATUS = {0: "HR_OK", 1: "HR_ERR_INVALID_ARG", 2: "HR_ERR_UNSUPPORTED", 3: "HR_ERR_WORKSPACE",
           4: "HR_ERR_CUDA", 5: "HR_ERR_NUMERIC"}


class hr_puncture(C.Structure):
    _fields_ = [("m", C.c_double), ("pos", C.c_double * 3), ("P", C.c_double * 3),
                ("S", C.c_double * 3)]


class hr_params(C.Structure):
    _fields_ = [
        ("n", C.c_int32 * 3),
        ("coord", C.c_int32),
        ("fd_order", C.c_int32),
        ("dtype", C.c_int32),
        ("amp", C.c_double),
        ("sinhw", C.c_double),
        ("bscale", C.c_double),
        ("origin", C.c_double * 3),
        ("n_punctures", C.c_int32),
        ("residual_mode", C.c_int32),
        ("punctures", C.POINTER(hr_puncture)),
        ("eta", C.c_double),
        ("cfl", C.c_double),
        ("c_min", C.c_double),
        ("device", C.c_int32),
        ("variant", C.c_int32),
        ("stream", C.c_void_p),
    ]


class HrError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"{_STATUS.get(status, status)}: {text}")
        self.status = status


if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'` "
        "(nvcc, sm_100a).  There is no CPU fallback.")

lib = C.CDLL(LIB_PATH)
_vp, _i32, _i64, _sz = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t
_SIGS = {
    "hr_workspace_bytes": [C.POINTER(hr_params), C.POINTER(_sz)],
    "hr_create": [C.POINTER(hr_params), _vp, _sz, C.POINTER(_vp)],
    "hr_destroy": [_vp],
    "hr_step": [_vp, _i64],
    "hr_residual": [_vp, C.POINTER(C.c_double)],
    "hr_residual_ex": [_vp, _i32, C.POINTER(C.c_double)],
    "hr_residual_async": [_vp, _i32, _vp],
    "hr_residual_static": [_vp, _i32, _vp],
    "hr_step_many": [C.POINTER(_vp), _i32, _i64],
    "hr_step_residual_async": [_vp, _i32, _vp],
    "hr_relax": [_vp, _i64, _i64, C.c_double, _i32, C.POINTER(_i64), C.POINTER(C.c_double), _vp, _i64,
                 C.POINTER(_i64)],
    "hr_get_u": [_vp, _vp, _sz, _i32],
    "hr_get_v": [_vp, _vp, _sz, _i32],
    "hr_set_state": [_vp, _vp, _vp, _i32],
    "hr_eval_rhs": [_vp, _vp, _vp],
    "hr_get_source": [_vp, _vp, _vp],
    "hr_get_bc_lists": [_vp, _vp, _vp, C.POINTER(_i64), _vp, C.POINTER(_i64)],
    "hr_get_info": [_vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(_i32),
                    C.POINTER(_i32), C.POINTER(_i64)],
    "hr_launches_per_step": [_vp, C.POINTER(_i32)],
    "hr_profile_step": [_vp, _i64, _i32, C.POINTER(C.c_double)],
    "hr_query": [_vp, _i32, C.POINTER(_i64)],
    "hr_measure_alu_peak": [_i32, _vp, _i32, _i32, C.POINTER(C.c_double)],
    "hr_measure_launch_floor": [_i32, _vp, _i32, _i32, _i32, _i32, C.POINTER(C.c_double)],
    "hr_host_setup": [C.POINTER(hr_params), C.POINTER(C.c_double), C.POINTER(C.c_double),
                      C.POINTER(_i64), C.POINTER(_i64), _vp, _vp, _vp, _vp, _vp],
}
for _name, _args in _SIGS.items():
    getattr(lib, _name).argtypes = _args
    getattr(lib, _name).restype = C.c_int
lib.hr_last_error.restype = C.c_char_p
lib.hr_version.restype = C.c_char_p


def _check(status):
    if status != HR_OK:
        raise HrError(status, lib.hr_last_error().decode())


def hr_step_many(solvers, n_steps: int):
    """n_steps RK4 steps of every Solver in `solvers`, interleaved, each on its own stream."""
    arr = (_vp * len(solvers))(*[s._h for s in solvers])
    _check(lib.hr_step_many(arr, _i32(len(solvers)), _i64(int(n_steps))))


HR_Q = {"step_graph": 0, "resid_graph": 1, "persistent": 2, "numeric_flag": 3, "plan_zc": 4, "plan_items": 5,
        "plan_grid": 6}


def hr_measure_alu_peak(dtype="f64", packed=False, device=0) -> float:
    """TFLOP/s of register-resident FMA chains (include/hr.h: hr_measure_alu_peak)."""
    import torch
    out = C.c_double()
    st = torch.cuda.current_stream(device).cuda_stream
    _check(lib.hr_measure_alu_peak(_i32(device), _vp(st), _i32(0 if dtype == "f64" else 1), _i32(int(packed)),
                                   C.byref(out)))
    return out.value


def hr_measure_launch_floor(nodes=4, grid=1, block=32, reps=200, device=0) -> float:
    """Microseconds per replay of a graph of `nodes` dependent empty launches (include/hr.h)."""
    import torch
    out = C.c_double()
    stream = torch.cuda.Stream(device)
    _check(lib.hr_measure_launch_floor(_i32(device), _vp(stream.cuda_stream), _i32(nodes), _i32(grid),
                                       _i32(block), _i32(reps), C.byref(out)))
    return out.value


def hr_version() -> str:
    return lib.hr_version().decode()


def make_params(params: dict, dtype="f64", device=0, stream=0, residual_mode=0, variant=0):
    """Neutral workload dict (hr_workloads) -> (hr_params, keep-alive puncture array)."""
    rows = np.asarray(params["punctures"], dtype=np.float64).reshape(-1, 10)
    punct = (hr_puncture * max(1, rows.shape[0]))()
    for q, r in enumerate(rows):
        punct[q].m = r[0]
        punct[q].pos[:] = r[1:4]
        punct[q].P[:] = r[4:7]
        punct[q].S[:] = r[7:10]
    p = hr_params()
    p.n[:] = [int(x) for x in params["n"]]
    p.coord = {"SinhSpherical": HR_SINHSPHERICAL, "SinhSymTP": HR_SINHSYMTP,
               "SinhCylindrical": HR_SINHCYLINDRICAL, "SinhCartesian": HR_SINHCARTESIAN}[params["coord"]]
    p.fd_order = int(params["fd_order"])
    p.dtype = {"f64": HR_F64, "f32": HR_F32}[dtype]
    p.amp = float(params["amp"])
    p.sinhw = float(params["sinhw"])
    p.bscale = float(params.get("bscale", 0.0))
    p.origin[:] = [float(x) for x in params.get("origin", (0.0, 0.0, 0.0))]
    p.n_punctures = int(rows.shape[0])
    p.residual_mode = int(residual_mode)
    p.punctures = C.cast(punct, C.POINTER(hr_puncture))
    p.eta = float(params["eta"])
    p.cfl = float(params["cfl"])
    p.c_min = float(params.get("c_min", 1.0))
    p.device = int(device)
    p.variant = int(variant)
    p.stream = C.c_void_p(int(stream))
    return p, punct


def hr_workspace_bytes(p: hr_params) -> int:
    n = _sz()
    _check(lib.hr_workspace_bytes(C.byref(p), C.byref(n)))
    return int(n.value)


def hr_host_setup(params: dict, dtype="f64") -> dict:
    """Host-only tables of hr_create (no device needed): dt, dsmin, boundary lists, planes."""
    p, _keep = make_params(params, dtype)
    dt, dsmin, ni, no = C.c_double(), C.c_double(), _i64(), _i64()
    _check(lib.hr_host_setup(C.byref(p), C.byref(dt), C.byref(dsmin), C.byref(ni), C.byref(no),
                             None, None, None, None, None))
    ng = p.fd_order // 2
    T = [p.n[a] + 2 * ng for a in range(3)]
    dst = np.empty(ni.value, np.int32)
    src = np.empty(ni.value, np.int32)
    out = np.empty(no.value, np.int32)
    planes = np.empty((7, T[1], T[0]))
    outer = np.empty((3, T[1], ng))
    _check(lib.hr_host_setup(C.byref(p), None, None, None, None, _vp(dst.ctypes.data),
                             _vp(src.ctypes.data), _vp(out.ctypes.data), _vp(planes.ctypes.data),
                             _vp(outer.ctypes.data)))
    names = ["L00", "L11", "L22", "L0", "L1", "C2", "W"]
    return dict(dt=dt.value, dsmin=dsmin.value, inner_dst=dst, inner_src=src, outer_idx=out, T=T,
                ng=ng, planes=dict(zip(names, planes)),
                outer=dict(zip(["RAD0", "RAD1", "RADI"], outer)))


class Solver:
    """hr_create / hr_step / hr_residual / hr_get_u / hr_get_v on one CUDA device.

    The workspace is a torch uint8 CUDA tensor owned by this object; work is enqueued on a
    dedicated torch stream (`self.stream`)."""

    def __init__(self, params: dict, dtype="f64", device=0, residual_mode=0, variant=0,
                 stream=None, poison=False):
        import torch  # device memory and streams only

        self._h = None
        if not torch.cuda.is_available():
            raise HrError(4, "no CUDA device: the hot path has no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.dtype = dtype
        self.tdtype = torch.float64 if dtype == "f64" else torch.float32
        self.npdtype = np.float64 if dtype == "f64" else np.float32
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        self.p, self._punct = make_params(params, dtype, device, self.stream.cuda_stream,
                                          residual_mode, variant)
        nbytes = hr_workspace_bytes(self.p)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        if poison:  # every byte 0xFF = NaN in both precisions: a read of workspace the library never wrote shows
            self.workspace.fill_(255)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        h = _vp()
        _check(lib.hr_create(C.byref(self.p), _vp(self._ws_ptr), _sz(nbytes), C.byref(h)))
        self._h = h
        dt, dsmin, ng, T, ntot = C.c_double(), C.c_double(), _i32(), (_i32 * 3)(), _i64()
        _check(lib.hr_get_info(h, C.byref(dt), C.byref(dsmin), C.byref(ng), T, C.byref(ntot)))
        self.dt, self.dsmin, self.ng = dt.value, dsmin.value, ng.value
        self.T = tuple(int(t) for t in T)
        self.n = tuple(int(x) for x in params["n"])
        self.ntot = int(ntot.value)
        self.n_int = self.n[0] * self.n[1] * self.n[2]
        self.workspace_bytes = nbytes
        n = _i32()
        _check(lib.hr_launches_per_step(h, C.byref(n)))
        self.launches_per_step = int(n.value)

    def close(self):
        if getattr(self, "_h", None):
            self.stream.synchronize()
            lib.hr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the calls of include/hr.h ----
    def hr_step(self, n_steps: int):
        _check(lib.hr_step(self._h, _i64(int(n_steps))))

    def hr_residual(self, mode=None) -> float:
        out = (C.c_double * 3)()
        m = self.p.residual_mode if mode is None else int(mode)
        _check(lib.hr_residual_ex(self._h, _i32(m), out))
        return float(out[0])

    def hr_residual_ex(self, mode):
        """(norm, sum w H^2, sum w) of the current state."""
        out = (C.c_double * 3)()
        _check(lib.hr_residual_ex(self._h, _i32(int(mode)), out))
        return float(out[0]), float(out[1]), float(out[2])

    def hr_residual_async(self, mode, out2):
        """out2: torch float64 CUDA tensor with >= 2 elements; receives {sum w H^2, sum w}."""
        _check(lib.hr_residual_async(self._h, _i32(int(mode)), _vp(out2.data_ptr())))

    def hr_residual_static(self, mode, out2):
        """hr_residual_async with the kernel's scratch in the library's static device array (no allocation)."""
        _check(lib.hr_residual_static(self._h, _i32(int(mode)), _vp(out2.data_ptr())))

    def hr_step_residual_async(self, mode, out2):
        """Residual of the current state into out2 (as hr_residual_async), then one RK4 step."""
        _check(lib.hr_step_residual_async(self._h, _i32(int(mode)), _vp(out2.data_ptr())))

    def _get(self, fn, to_host):
        t = self.torch
        if to_host:
            out = np.empty(self.ntot, dtype=self.npdtype)
            _check(fn(self._h, _vp(out.ctypes.data), _sz(out.nbytes), _i32(0)))
            return out
        out = t.empty(self.ntot, dtype=self.tdtype, device=self.device)
        _check(fn(self._h, _vp(out.data_ptr()), _sz(out.numel() * out.element_size()), _i32(1)))
        return out

    def hr_get_u(self, to_host=True):
        return self._get(lib.hr_get_u, to_host)

    def hr_get_v(self, to_host=True):
        return self._get(lib.hr_get_v, to_host)

    def hr_set_state(self, u, v):
        """u, v: numpy arrays (host) or torch CUDA tensors (device) of N_tot scalars."""
        if isinstance(u, np.ndarray):
            u = np.ascontiguousarray(u, dtype=self.npdtype)
            v = np.ascontiguousarray(v, dtype=self.npdtype)
            assert u.size == self.ntot and v.size == self.ntot
            _check(lib.hr_set_state(self._h, _vp(u.ctypes.data), _vp(v.ctypes.data), _i32(0)))
        else:
            assert u.is_cuda and u.dtype == self.tdtype and u.numel() == self.ntot
            # order the copy after whatever produced u, v on the caller's current stream
            self.stream.wait_stream(self.torch.cuda.current_stream(self.device))
            _check(lib.hr_set_state(self._h, _vp(u.data_ptr()), _vp(v.data_ptr()), _i32(1)))

    def hr_set_state_pinned(self, u_pinned, v_pinned):
        """u, v: pinned host torch tensors; asynchronous H2D is still followed by a stream sync
        inside hr_set_state (host source)."""
        _check(lib.hr_set_state(self._h, _vp(u_pinned.data_ptr()), _vp(v_pinned.data_ptr()), _i32(0)))

    def hr_eval_rhs(self):
        t = self.torch
        ku = t.empty(self.ntot, dtype=self.tdtype, device=self.device)
        kv = t.empty(self.ntot, dtype=self.tdtype, device=self.device)
        _check(lib.hr_eval_rhs(self._h, _vp(ku.data_ptr()), _vp(kv.data_ptr())))
        self.stream.synchronize()
        return ku.cpu().numpy(), kv.cpu().numpy()

    def hr_get_source(self):
        psi = np.empty(self.ntot, dtype=self.npdtype)
        S = np.empty(self.ntot, dtype=self.npdtype)
        _check(lib.hr_get_source(self._h, _vp(psi.ctypes.data), _vp(S.ctypes.data)))
        return psi, S

    def hr_get_bc_lists(self):
        ni, no = _i64(), _i64()
        _check(lib.hr_get_bc_lists(self._h, None, None, C.byref(ni), None, C.byref(no)))
        dst = np.empty(ni.value, dtype=np.int32)
        src = np.empty(ni.value, dtype=np.int32)
        out = np.empty(no.value, dtype=np.int32)
        _check(lib.hr_get_bc_lists(self._h, _vp(dst.ctypes.data), _vp(src.ctypes.data), C.byref(ni),
                                   _vp(out.ctypes.data), C.byref(no)))
        return dst, src, out

    def hr_relax(self, max_steps: int, check_every: int, tol: float, mode=0):
        """Alg. 1's relaxation loop with stopping criterion -> (steps done, final residual, history)."""
        cap = int(max_steps) // max(1, int(check_every)) + 3
        hist = np.zeros(cap, dtype=np.float64)
        done, nh, res = _i64(0), _i64(0), C.c_double(0.0)
        _check(lib.hr_relax(self._h, _i64(int(max_steps)), _i64(int(check_every)), C.c_double(float(tol)),
                            _i32(int(mode)), C.byref(done), C.byref(res), _vp(hist.ctypes.data), _i64(cap),
                            C.byref(nh)))
        return int(done.value), float(res.value), hist[:min(cap, int(nh.value))].copy()

    def hr_query(self, what: str) -> int:
        out = _i64()
        _check(lib.hr_query(self._h, _i32(HR_Q[what]), C.byref(out)))
        return out.value

    def hr_profile_step(self, n_steps: int, with_residual=True):
        """Mean ms per RK4 step in {stage 1..4 fused kernel, inner fills, residual}."""
        out = (C.c_double * 6)()
        _check(lib.hr_profile_step(self._h, _i64(int(n_steps)), _i32(int(bool(with_residual))), out))
        return [float(x) for x in out]

    def synchronize(self):
        self.stream.synchronize()
