"""Thin ctypes binding of include/catapult.h: argument marshalling only.

Every step of the path runs in the kernels of libcatapult.so.  PyTorch supplies device memory
(tensor.data_ptr()) and the current CUDA stream; numpy arrays are accepted by the *_host calls.
The library is loaded from the package directory and the import fails loudly when it is missing
(there is no CPU fallback; the oracle under oracle/ is test infrastructure and never used here).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libcatapult.so")
PROBE_LIB_PATH = os.path.join(_PKG, "libcatapult_probe.so")

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED = 0, 1, 2, 3, 4
COORD_BOOZER, COORD_CYL = 0, 1
ST_REACHED_T, ST_LOST, ST_STALLED, ST_MAXSTEPS = 0, 1, 2, 3
NCOUNTERS = 10
COUNTER_NAMES = ["accepted", "rejected", "reached_T", "lost", "stalled", "max_steps", "rhs_evals", "cell_fetches",
                 "blocking_fetches", "rounds"]

EXPORTS = [
    "catapult_field_build", "catapult_field_build_host", "catapult_field_destroy",
    "catapult_field_table_bytes", "catapult_field_eval", "catapult_field_export_rows",
    "catapult_trace", "catapult_trace_init", "catapult_trace_continue", "catapult_trace_host",
    "catapult_trace_continue_host", "catapult_release_host_cache", "catapult_trace_scripted",
    "catapult_step_once", "catapult_estimate", "catapult_estimate_static", "catapult_measure_lost_energy",
    "catapult_exit_histogram", "catapult_trace_launch_shape", "catapult_last_error",
    "catapult_version",
]
PROBE_EXPORTS = ["catapult_math_probe", "catapult_measure_fp64_peak", "catapult_measure_l2_bandwidth",
                 "catapult_probe_last_error"]


class FieldDesc(C.Structure):
    _fields_ = [("coord", C.c_int32), ("ncell", C.c_int32 * 3), ("nfp", C.c_int32),
                ("nquant", C.c_int32), ("quant", C.c_int32 * 16), ("lo", C.c_double * 3), ("hi", C.c_double * 3),
                ("G0", C.c_double), ("I0", C.c_double), ("iota0", C.c_double),
                ("iota1", C.c_double), ("psi0", C.c_double), ("G_nodes", C.c_void_p), ("I_nodes", C.c_void_p),
                ("iota_nodes", C.c_void_p)]


class TraceParams(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("energy", C.c_double),
                ("T", C.c_double), ("rtol", C.c_double), ("atol", C.c_double),
                ("dt0", C.c_double), ("dtmax", C.c_double), ("max_steps", C.c_int64),
                ("max_consecutive_rejects", C.c_int32), ("saw_on", C.c_int32),
                ("saw_m", C.c_int32), ("saw_n", C.c_int32), ("saw_Phi0", C.c_double),
                ("saw_s0", C.c_double), ("saw_w2", C.c_double), ("saw_omega", C.c_double),
                ("loss_time_mode", C.c_int32), ("reserved_", C.c_int32)]


class CatapultError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"catapult status {status}: {message}")
        self.status = status


_lib = None
_probe = None


def load():
    """Loads libcatapult.so (building is __graft_entry__.build()'s job) -- loud failure if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2604_07617_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, dp = C.c_void_p, C.c_int64, C.c_void_p
    L.catapult_field_build.argtypes = [C.POINTER(FieldDesc), dp, vp, C.POINTER(vp)]
    L.catapult_field_build_host.argtypes = [C.POINTER(FieldDesc), dp, C.POINTER(vp)]
    L.catapult_field_destroy.argtypes = [vp]
    L.catapult_field_table_bytes.argtypes = [vp]
    L.catapult_field_table_bytes.restype = C.c_size_t
    L.catapult_field_eval.argtypes = [vp, i64, dp, dp, vp]
    L.catapult_field_export_rows.argtypes = [vp, dp, vp]
    L.catapult_trace.argtypes = [vp, C.POINTER(TraceParams), i64, dp, dp, dp, dp, dp, dp, dp, vp]
    L.catapult_trace_init.argtypes = [vp, C.POINTER(TraceParams), i64, dp, dp, dp, dp, dp, vp]
    L.catapult_trace_continue.argtypes = [vp, C.POINTER(TraceParams), i64, dp, dp, dp, dp, dp, dp, dp, dp, vp]
    L.catapult_trace_host.argtypes = [vp, C.POINTER(TraceParams), i64, dp, dp, dp, dp, dp, dp, dp]
    L.catapult_trace_continue_host.argtypes = [vp, C.POINTER(TraceParams), i64, dp, dp, dp, dp, dp, dp, dp, dp]
    L.catapult_trace_scripted.argtypes = [vp, C.POINTER(TraceParams), i64, dp, C.c_int32, dp, dp, dp, dp, dp, vp]
    L.catapult_step_once.argtypes = [vp, C.POINTER(TraceParams), i64, dp, dp, dp, dp, dp, dp, vp]
    L.catapult_estimate.argtypes = [C.c_int32, i64, dp, dp, dp, dp, dp, vp]
    L.catapult_estimate_static.argtypes = [C.c_int32, i64, dp, dp, dp, dp, vp]
    L.catapult_measure_lost_energy.argtypes = [vp, C.POINTER(TraceParams), i64, dp, dp, dp, dp, vp]
    L.catapult_exit_histogram.argtypes = [vp, i64, dp, dp, C.c_int32, C.c_int32, dp, vp]
    L.catapult_release_host_cache.argtypes = []
    L.catapult_trace_launch_shape.argtypes = [vp, C.POINTER(TraceParams), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.catapult_last_error.restype = C.c_char_p
    L.catapult_version.restype = C.c_char_p
    for name in EXPORTS:
        fn = getattr(L, name)
        if fn.restype is C.c_int:
            fn.restype = C.c_int
    _lib = L
    return L


def load_probe():
    """Loads libcatapult_probe.so: measurement / test hooks (include/catapult_probe.h), not the product."""
    global _probe
    if _probe is not None:
        return _probe
    if not os.path.exists(PROBE_LIB_PATH):
        raise ImportError(f"{PROBE_LIB_PATH} is missing: run `python -m paper_2604_07617_b200.build`")
    P = C.CDLL(PROBE_LIB_PATH)
    dp = C.c_void_p
    P.catapult_math_probe.argtypes = [C.c_int32, C.c_int64, dp, dp, dp, dp, C.c_void_p]
    P.catapult_measure_fp64_peak.argtypes = [C.POINTER(C.c_double)]
    P.catapult_measure_l2_bandwidth.argtypes = [C.c_size_t, C.POINTER(C.c_double)]
    P.catapult_probe_last_error.restype = C.c_char_p
    _probe = P
    return P


def _check(st: int):
    if st != OK:
        raise CatapultError(st, load().catapult_last_error().decode())


def _check_probe(st: int):
    if st != OK:
        raise CatapultError(st, load_probe().catapult_probe_last_error().decode())


def make_desc(fd: dict) -> FieldDesc:
    d = FieldDesc()
    d.coord = int(fd["coord"])
    for i in range(3):
        d.ncell[i] = int(fd["ncell"][i])
        d.lo[i] = float(fd["lo"][i])
        d.hi[i] = float(fd["hi"][i])
    d.nfp = int(fd["nfp"])
    d.nquant = int(fd["nquant"])
    for k in ("G0", "I0", "iota0", "iota1", "psi0"):
        setattr(d, k, float(fd.get(k, 0.0)))
    for i, tag in enumerate(fd.get("quant", ())):
        d.quant[i] = int(tag)
    keep = []
    for k in ("G_nodes", "I_nodes", "iota_nodes"):        # CUDA tensors (device pointers), numpy arrays, or absent
        t = fd.get(k)
        if t is None:
            setattr(d, k, None)
        elif isinstance(t, np.ndarray):                    # host array: the library copies it (any direction)
            t = np.ascontiguousarray(t, dtype=np.float64)
            keep.append(t)
            setattr(d, k, t.ctypes.data)
        else:
            keep.append(t)
            setattr(d, k, t.data_ptr())
    d._keep = keep                                         # alive until the build call has returned
    return d


def make_params(pd: dict) -> TraceParams:
    p = TraceParams()
    for name, _ in TraceParams._fields_:
        if name in pd:
            setattr(p, name, pd[name])
    return p


def _torch():
    import torch
    return torch


def _stream():
    return C.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _ptr(t, dtype=None, allow_none=False):
    """device pointer of a contiguous CUDA tensor"""
    if t is None:
        if allow_none:
            return None
        raise ValueError("required tensor is None")
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _hptr(a, dtype):
    if a is None:
        return None
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags["C_CONTIGUOUS"]):
        raise TypeError(f"expected a C-contiguous numpy array of {dtype}")
    return C.c_void_p(a.ctypes.data)


class Field:
    """Owns a catapult_field (the per-cell coefficient tables on the device)."""

    def __init__(self, handle, desc: FieldDesc):
        self._h = handle
        self.desc = desc

    @property
    def nquant(self) -> int:
        return int(self.desc.nquant)

    @property
    def ncells(self) -> int:
        return int(self.desc.ncell[0]) * int(self.desc.ncell[1]) * int(self.desc.ncell[2])

    @property
    def table_bytes(self) -> int:
        return int(load().catapult_field_table_bytes(self._h))

    def destroy(self):
        if self._h is not None:
            load().catapult_field_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def catapult_field_build(fd: dict, d_nodes=None) -> Field:
    """fd: field dict (workloads.py); d_nodes: CUDA float64 tensor [m][n0][n1][n2] (default: fd['nodes']
    uploaded with torch)."""
    L = load()
    torch = _torch()
    desc = make_desc(fd)
    if d_nodes is None:
        d_nodes = torch.from_numpy(np.ascontiguousarray(fd["nodes"], dtype=np.float64)).cuda()
    n = [3 * int(k) + 1 for k in fd["ncell"]]
    if tuple(d_nodes.shape) != (desc.nquant, n[0], n[1], n[2]):
        raise ValueError(f"nodes shape {tuple(d_nodes.shape)} != {(desc.nquant, *n)}")
    h = C.c_void_p()
    _check(L.catapult_field_build(C.byref(desc), _ptr(d_nodes, torch.float64), _stream(), C.byref(h)))
    return Field(h, desc)


def catapult_field_build_host(fd: dict) -> Field:
    L = load()
    desc = make_desc(fd)
    nodes = np.ascontiguousarray(fd["nodes"], dtype=np.float64)
    h = C.c_void_p()
    _check(L.catapult_field_build_host(C.byref(desc), _hptr(nodes, np.float64), C.byref(h)))
    return Field(h, desc)


def catapult_field_eval(f: Field, d_pts):
    torch = _torch()
    npts = d_pts.shape[1]
    out = torch.empty((f.nquant, npts), dtype=torch.float64, device=d_pts.device)
    _check(load().catapult_field_eval(f._h, npts, _ptr(d_pts, torch.float64), _ptr(out), _stream()))
    return out


def catapult_field_export_rows(f: Field):
    torch = _torch()
    out = torch.empty((f.ncells * 64, f.nquant), dtype=torch.float64, device="cuda")
    _check(load().catapult_field_export_rows(f._h, _ptr(out), _stream()))
    return out


def catapult_trace(f: Field, pd: dict, d_x0, counters: bool = True) -> dict:
    """Traces d_x0 [4][n] (CUDA float64) from t=0 to min(tau,T).  Returns device tensors."""
    torch = _torch()
    p = make_params(pd)
    n = d_x0.shape[1]
    dev = d_x0.device
    xf = torch.empty((4, n), dtype=torch.float64, device=dev)
    tstop = torch.empty(n, dtype=torch.float64, device=dev)
    status = torch.empty(n, dtype=torch.int32, device=dev)
    nacc = torch.empty(n, dtype=torch.int32, device=dev)
    nrej = torch.empty(n, dtype=torch.int32, device=dev)
    cnt = torch.zeros(NCOUNTERS, dtype=torch.int64, device=dev) if counters else None
    _check(load().catapult_trace(f._h, C.byref(p), n, _ptr(d_x0, torch.float64), _ptr(xf), _ptr(tstop),
                                 _ptr(status), _ptr(nacc), _ptr(nrej), _ptr(cnt, allow_none=True), _stream()))
    return dict(xf=xf, tstop=tstop, status=status, nacc=nacc, nrej=nrej, counters=cnt)


def catapult_trace_init(f: Field, pd: dict, d_x) -> dict:
    torch = _torch()
    p = make_params(pd)
    n = d_x.shape[1]
    dev = d_x.device
    st = dict(x=d_x, t=torch.empty(n, dtype=torch.float64, device=dev),
              dt=torch.empty(n, dtype=torch.float64, device=dev),
              mu=torch.empty(n, dtype=torch.float64, device=dev),
              status=torch.empty(n, dtype=torch.int32, device=dev),
              nacc=torch.zeros(n, dtype=torch.int32, device=dev),
              nrej=torch.zeros(n, dtype=torch.int32, device=dev),
              counters=torch.zeros(NCOUNTERS, dtype=torch.int64, device=dev))
    _check(load().catapult_trace_init(f._h, C.byref(p), n, _ptr(d_x, torch.float64), _ptr(st["t"]), _ptr(st["dt"]),
                                      _ptr(st["mu"]), _ptr(st["status"]), _stream()))
    return st


def catapult_trace_continue(f: Field, pd: dict, st: dict) -> dict:
    """Advances the in/out state dict of catapult_trace_init to pd['T'] (in place)."""
    torch = _torch()
    p = make_params(pd)
    n = st["x"].shape[1]
    _check(load().catapult_trace_continue(f._h, C.byref(p), n, _ptr(st["x"], torch.float64), _ptr(st["t"]),
                                          _ptr(st["dt"]), _ptr(st["mu"]), _ptr(st["status"]), _ptr(st["nacc"]),
                                          _ptr(st["nrej"]), _ptr(st["counters"]), _stream()))
    return st


def catapult_trace_host(f: Field, pd: dict, h_x0: np.ndarray, out: dict | None = None) -> dict:
    """HOST-buffer trace: numpy in, numpy out; H2D and D2H copies happen inside the call."""
    p = make_params(pd)
    n = h_x0.shape[1]
    if out is None:
        out = dict(xf=np.empty((4, n)), tstop=np.empty(n), status=np.empty(n, dtype=np.int32),
                   nacc=np.empty(n, dtype=np.uint32), nrej=np.empty(n, dtype=np.uint32),
                   counters=np.zeros(NCOUNTERS, dtype=np.uint64))
    _check(load().catapult_trace_host(f._h, C.byref(p), n, _hptr(h_x0, np.float64), _hptr(out["xf"], np.float64),
                                      _hptr(out["tstop"], np.float64), _hptr(out["status"], np.int32),
                                      _hptr(out["nacc"], np.uint32), _hptr(out["nrej"], np.uint32),
                                      _hptr(out["counters"], np.uint64)))
    return out


def catapult_trace_continue_host(f: Field, pd: dict, st: dict) -> dict:
    """HOST-buffer continue: st holds numpy arrays x[4][n], t, dt, mu (float64), status (int32),
    nacc, nrej (uint32), counters (uint64[NCOUNTERS]); all updated in place."""
    p = make_params(pd)
    n = st["x"].shape[1]
    _check(load().catapult_trace_continue_host(
        f._h, C.byref(p), n, _hptr(st["x"], np.float64), _hptr(st["t"], np.float64), _hptr(st["dt"], np.float64),
        _hptr(st["mu"], np.float64), _hptr(st["status"], np.int32), _hptr(st.get("nacc"), np.uint32),
        _hptr(st.get("nrej"), np.uint32), _hptr(st.get("counters"), np.uint64)))
    return st


def catapult_trace_scripted(f: Field, pd: dict, d_x0, d_h) -> dict:
    """Replays the step sizes d_h [nsteps][n] (CUDA float64) from d_x0 [4][n]; every step is accepted."""
    torch = _torch()
    p = make_params(pd)
    n = d_x0.shape[1]
    nsteps = d_h.shape[0]
    dev = d_x0.device
    xf = torch.empty((4, n), dtype=torch.float64, device=dev)
    tstop = torch.empty(n, dtype=torch.float64, device=dev)
    status = torch.empty(n, dtype=torch.int32, device=dev)
    r = torch.full((nsteps, n), float("nan"), dtype=torch.float64, device=dev)
    _check(load().catapult_trace_scripted(f._h, C.byref(p), n, _ptr(d_x0, torch.float64), nsteps,
                                          _ptr(d_h, torch.float64), _ptr(xf), _ptr(tstop), _ptr(status), _ptr(r),
                                          _stream()))
    return dict(xf=xf, tstop=tstop, status=status, r=r)


def catapult_step_once(f: Field, pd: dict, d_x, d_t, d_h):
    torch = _torch()
    p = make_params(pd)
    n = d_x.shape[1]
    dev = d_x.device
    xnew = torch.empty((4, n), dtype=torch.float64, device=dev)
    err = torch.empty(n, dtype=torch.float64, device=dev)
    k = torch.empty((7, 4, n), dtype=torch.float64, device=dev)
    _check(load().catapult_step_once(f._h, C.byref(p), n, _ptr(d_x, torch.float64), _ptr(d_t, torch.float64),
                                     _ptr(d_h, torch.float64), _ptr(xnew), _ptr(err), _ptr(k), _stream()))
    return xnew, err, k


def catapult_estimate(g_kind: int, d_status=None, d_tstop=None, d_g_user=None, to_host: bool = True):
    """Returns (mean, standard error, sum g, sum g^2) -- numpy[4] when to_host else a CUDA tensor."""
    torch = _torch()
    ref = d_status if d_status is not None else (d_tstop if d_tstop is not None else d_g_user)
    n = ref.shape[0]
    out = torch.empty(4, dtype=torch.float64, device=ref.device)
    h = np.zeros(4) if to_host else None
    _check(load().catapult_estimate(g_kind, n, _ptr(d_status, torch.int32, True), _ptr(d_tstop, torch.float64, True),
                                    _ptr(d_g_user, torch.float64, True), _ptr(out), _hptr(h, np.float64), _stream()))
    return h if to_host else out


def catapult_measure_lost_energy(f: Field, pd: dict, d_xf, d_mu, d_status):
    """g[i] = 1[lost] (vpar^2/2 + mu |B|(x_f)) / (v_total^2/2) as a CUDA float64[n] tensor (feed it to
    catapult_estimate(2, d_g_user=g))."""
    torch = _torch()
    p = make_params(pd)
    n = d_xf.shape[1]
    g = torch.empty(n, dtype=torch.float64, device=d_xf.device)
    _check(load().catapult_measure_lost_energy(f._h, C.byref(p), n, _ptr(d_xf, torch.float64), _ptr(d_mu, torch.float64),
                                               _ptr(d_status, torch.int32), _ptr(g), _stream()))
    return g


def catapult_exit_histogram(f: Field, d_xf, d_status, nbins0: int, nbins1: int):
    """Lost particles per bin of the exit point: CUDA int64[nbins0][nbins1]."""
    torch = _torch()
    n = d_xf.shape[1]
    hist = torch.empty((nbins0, nbins1), dtype=torch.int64, device=d_xf.device)
    _check(load().catapult_exit_histogram(f._h, n, _ptr(d_xf, torch.float64), _ptr(d_status, torch.int32), nbins0, nbins1,
                                          _ptr(hist), _stream()))
    return hist


ESTIMATE_STATIC_MAX_N = 2097152


def catapult_estimate_static(g_kind: int, d_status=None, d_tstop=None, d_g_user=None, out=None):
    """catapult_estimate for callers that must not allocate device memory (a process whose GPU memory is owned by its
    own manager, a latency-bound loop, a driver without memory pools): same four numbers, bit-identical, with the
    partial sums in a 16 KiB array built into the library instead of a stream-ordered allocation.

    `out` is the caller's CUDA float64[4] result tensor, filled on the current stream and returned (nothing is copied
    to the host).  Pass it: when it is omitted this wrapper makes one with torch.empty, which allocates -- fine in a
    test, not what a no-allocation caller wants.  At most ESTIMATE_STATIC_MAX_N particles (CatapultError otherwise).
    All calls on a GPU share the array: keep them on one stream or order them yourself.  The first call on a device
    looks the array up; make it during set-up."""
    torch = _torch()
    ref = d_status if d_status is not None else (d_tstop if d_tstop is not None else d_g_user)
    n = ref.shape[0]
    if out is None:
        out = torch.empty(4, dtype=torch.float64, device=ref.device)
    _check(load().catapult_estimate_static(g_kind, n, _ptr(d_status, torch.int32, True),
                                           _ptr(d_tstop, torch.float64, True), _ptr(d_g_user, torch.float64, True),
                                           _ptr(out, torch.float64), _stream()))
    return out


FN_ATAN2, FN_SINCOS, FN_EXP, FN_SQRT_RSQRT, FN_RCP, FN_POW_NEG_INV, FN_CONTROLLER = range(7)


def catapult_math_probe(fn: int, d_a, d_b=None):
    """Test hook: (out0, out1) of the device-side elementary function `fn` on CUDA float64 tensors."""
    torch = _torch()
    o0, o1 = torch.empty_like(d_a), torch.empty_like(d_a)
    _check_probe(load_probe().catapult_math_probe(fn, d_a.numel(), _ptr(d_a, torch.float64),
                                                  _ptr(d_b, torch.float64, True), _ptr(o0), _ptr(o1), _stream()))
    return o0, o1


def catapult_measure_fp64_peak() -> float:
    v = C.c_double(0)
    _check_probe(load_probe().catapult_measure_fp64_peak(C.byref(v)))
    return v.value


def catapult_measure_l2_bandwidth(nbytes: int) -> float:
    v = C.c_double(0)
    _check_probe(load_probe().catapult_measure_l2_bandwidth(nbytes, C.byref(v)))
    return v.value


def catapult_release_host_cache():
    _check(load().catapult_release_host_cache())


def catapult_trace_launch_shape(f: Field, pd: dict):
    p = make_params(pd)
    b, t = C.c_int32(0), C.c_int32(0)
    _check(load().catapult_trace_launch_shape(f._h, C.byref(p), C.byref(b), C.byref(t)))
    return b.value, t.value
