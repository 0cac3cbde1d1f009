"""ctypes front-end of the plain C oracle (oracle/catapult_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: imported only by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  Argument marshalling only; all arithmetic is
in the C file, which cites PAPER.md passage by passage.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_c_double_p = C.POINTER(C.c_double)
ANALYTIC_FN = C.CFUNCTYPE(None, C.c_void_p, _c_double_p, _c_double_p)
ODE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_double, _c_double_p, _c_double_p)


class CField(C.Structure):
    _fields_ = [
        ("coord", C.c_int32), ("ncell", C.c_int32 * 3), ("nfp", C.c_int32), ("nquant", C.c_int32),
        ("lo", C.c_double * 3), ("hi", C.c_double * 3),
        ("nodes", _c_double_p),
        ("G0", C.c_double), ("I0", C.c_double), ("iota0", C.c_double), ("iota1", C.c_double),
        ("psi0", C.c_double),
        ("analytic", ANALYTIC_FN), ("analytic_ctx", C.c_void_p),
        ("G_nodes", _c_double_p), ("I_nodes", _c_double_p), ("iota_nodes", _c_double_p),
    ]


class CParams(C.Structure):
    _fields_ = [
        ("mass", C.c_double), ("charge", C.c_double), ("energy", C.c_double),
        ("T", C.c_double), ("rtol", C.c_double), ("atol", C.c_double),
        ("dt0", C.c_double), ("dtmax", C.c_double),
        ("max_steps", C.c_int64), ("max_consecutive_rejects", C.c_int32),
        ("saw_on", C.c_int32), ("saw_m", C.c_int32), ("saw_n", C.c_int32),
        ("saw_Phi0", C.c_double), ("saw_s0", C.c_double), ("saw_w2", C.c_double),
        ("saw_omega", C.c_double),
        ("loss_time_mode", C.c_int32), ("reserved_", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        L = _lib
        L.orc_vtotal.restype = C.c_double
        L.orc_mu_init.restype = C.c_double
        L.orc_error_ratio.restype = C.c_double
        L.orc_controller.restype = C.c_double
        L.orc_trace_record.restype = C.c_int64
        L.orc_trace_scripted.restype = C.c_int64
        L.orc_max_threads.restype = C.c_int
        L.orc_loss_refine.restype = C.c_double
    return _lib


def _dp(a):
    return a.ctypes.data_as(_c_double_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Field:
    """Wraps a field dict from paper_2604_07617_b200.workloads (or an analytic callback)."""

    def __init__(self, fd: dict, analytic=None):
        self.fd = fd
        self.c = CField()
        self.c.coord = int(fd["coord"])
        for d in range(3):
            self.c.ncell[d] = int(fd["ncell"][d])
            self.c.lo[d] = float(fd["lo"][d])
            self.c.hi[d] = float(fd["hi"][d])
        self.c.nfp = int(fd["nfp"])
        self.c.nquant = int(fd["nquant"])
        self.nodes = None
        if fd.get("nodes") is not None:
            self.nodes = _f64(fd["nodes"])
            n = [3 * int(k) + 1 for k in fd["ncell"]]
            assert self.nodes.shape == (self.c.nquant, n[0], n[1], n[2]), self.nodes.shape
            self.c.nodes = _dp(self.nodes)
        for k in ("G0", "I0", "iota0", "iota1", "psi0"):
            setattr(self.c, k, float(fd.get(k, 0.0)))
        self.profiles = {}
        for k in ("G_nodes", "I_nodes", "iota_nodes"):   # non-vacuum Boozer: profiles on the unique s-nodes
            if fd.get(k) is not None:
                self.profiles[k] = _f64(fd[k])
                assert self.profiles[k].shape == (3 * int(fd["ncell"][0]) + 1,), self.profiles[k].shape
                setattr(self.c, k, _dp(self.profiles[k]))
        self._cb = None
        if analytic is not None:
            m = self.c.nquant

            def _cb(_ctx, xp, outp):
                vals = analytic(np.array([xp[0], xp[1], xp[2]]))
                for q in range(m):
                    outp[q] = float(vals[q])

            self._cb = ANALYTIC_FN(_cb)
            self.c.analytic = self._cb

    @property
    def ref(self):
        return C.byref(self.c)


def make_params(pd: dict) -> CParams:
    p = CParams()
    for name, _ in CParams._fields_:
        if name in pd:
            setattr(p, name, pd[name])
    return p


# ---- thin calls ---------------------------------------------------------------------------
def lagrange4(u: float) -> np.ndarray:
    L = np.zeros(4)
    lib().orc_lagrange4(C.c_double(u), _dp(L))
    return L


def locate(f: Field, x):
    x = _f64(x)
    cell = np.zeros(3, dtype=np.int32)
    u = np.zeros(3)
    lib().orc_locate(f.ref, _dp(x), cell.ctypes.data_as(C.POINTER(C.c_int32)), _dp(u))
    return cell, u


def tricubic(f: Field, x) -> np.ndarray:
    x = _f64(x)
    out = np.zeros(16)
    lib().orc_tricubic(f.ref, _dp(x), _dp(out))
    return out[: f.c.nquant].copy()


def tricubic_many(f: Field, pts) -> np.ndarray:
    pts = _f64(pts)
    assert pts.ndim == 2 and pts.shape[0] == 3
    n = pts.shape[1]
    out = np.zeros((f.c.nquant, n))
    lib().orc_tricubic_many(f.ref, C.c_int64(n), _dp(pts), _dp(out))
    return out


def field_build(f: Field) -> np.ndarray:
    k = [int(v) for v in f.fd["ncell"]]
    out = np.zeros((k[0] * k[1] * k[2] * 64, f.c.nquant))
    lib().orc_field_build(f.ref, _dp(out))
    return out


def gc_boozer(f: Field, p: CParams, mu, t, s, theta, zeta, vpar, fv) -> np.ndarray:
    fv = _f64(fv)
    out = np.zeros(4)
    lib().orc_gc_boozer(f.ref, C.byref(p), C.c_double(mu), C.c_double(t), C.c_double(s),
                        C.c_double(theta), C.c_double(zeta), C.c_double(vpar), _dp(fv), _dp(out))
    return out


def gc_cartesian(p: CParams, mu, pos, vpar, fv) -> np.ndarray:
    pos = _f64(pos)
    fv = _f64(fv)
    out = np.zeros(4)
    lib().orc_gc_cartesian(C.byref(p), C.c_double(mu), _dp(pos), C.c_double(vpar), _dp(fv),
                           _dp(out))
    return out


def rhs(f: Field, p: CParams, mu, t, y):
    y = _f64(y)
    dy = np.zeros(4)
    fv = np.zeros(16)
    lib().orc_rhs(f.ref, C.byref(p), C.c_double(mu), C.c_double(t), _dp(y), _dp(dy), _dp(fv))
    return dy, fv[: (4 if f.c.nquant == 1 else f.c.nquant)].copy()


def dp5_tableau():
    c = np.zeros(7)
    a = np.zeros((7, 7))
    b = np.zeros(7)
    e = np.zeros(7)
    lib().orc_dp5_tableau(_dp(c), _dp(a), _dp(b), _dp(e))
    return c, a, b, e


def dp5_attempt(fun, t, y, h):
    """fun(t, y)->dy python callable; returns ynew, k7, err, kall[7][n]."""
    y = _f64(y)
    n = y.size

    def _cb(_ctx, tt, yp, dyp):
        d = fun(tt, np.array([yp[i] for i in range(n)]))
        for i in range(n):
            dyp[i] = float(d[i])

    cb = ODE_FN(_cb)
    k1 = _f64(fun(t, y))
    ynew = np.zeros(n)
    k7 = np.zeros(n)
    err = np.zeros(n)
    kall = np.zeros((7, n))
    lib().orc_dp5_attempt(cb, None, C.c_int(n), C.c_double(t), _dp(y), _dp(k1), C.c_double(h),
                          _dp(ynew), _dp(k7), _dp(err), _dp(kall))
    return ynew, k7, err, kall


def error_ratio(err, y, k1, h, rtol, atol, cscale) -> float:
    err, y, k1, cscale = _f64(err), _f64(y), _f64(k1), _f64(cscale)
    return float(lib().orc_error_ratio(C.c_int(err.size), _dp(err), _dp(y), _dp(k1), C.c_double(h),
                                       C.c_double(rtol), C.c_double(atol), _dp(cscale)))


def controller(h, r, dtmax):
    acc = C.c_int(0)
    dt = lib().orc_controller(C.c_double(h), C.c_double(r), C.c_double(dtmax), C.byref(acc))
    return float(dt), bool(acc.value)


def vtotal(p: CParams) -> float:
    return float(lib().orc_vtotal(C.byref(p)))


def default_steps(f: Field, p: CParams):
    a = C.c_double(0)
    b = C.c_double(0)
    lib().orc_default_steps(f.ref, C.byref(p), C.byref(a), C.byref(b))
    return a.value, b.value


def mu_init(f: Field, p: CParams, x) -> float:
    x = _f64(x)
    return float(lib().orc_mu_init(f.ref, C.byref(p), _dp(x)))


def trace(f: Field, p: CParams, x0, nthreads: int = 0):
    x0 = _f64(x0)
    assert x0.ndim == 2 and x0.shape[0] == 4
    n = x0.shape[1]
    xf = np.zeros((4, n))
    tstop = np.zeros(n)
    status = np.zeros(n, dtype=np.int32)
    nacc = np.zeros(n, dtype=np.uint32)
    nrej = np.zeros(n, dtype=np.uint32)
    lib().orc_trace(f.ref, C.byref(p), C.c_int64(n), _dp(x0), _dp(xf), _dp(tstop),
                    status.ctypes.data_as(C.POINTER(C.c_int32)),
                    nacc.ctypes.data_as(C.POINTER(C.c_uint32)),
                    nrej.ctypes.data_as(C.POINTER(C.c_uint32)), C.c_int(nthreads))
    return dict(xf=xf, tstop=tstop, status=status, nacc=nacc, nrej=nrej)


def step_once(f: Field, p: CParams, x, t, h):
    x = _f64(x)
    xnew = np.zeros(4)
    r = C.c_double(0)
    k = np.zeros((7, 4))
    lib().orc_step_once(f.ref, C.byref(p), _dp(x), C.c_double(t), C.c_double(h), _dp(xnew),
                        C.byref(r), _dp(k))
    return xnew, r.value, k


def trace_record(f: Field, p: CParams, x0, maxrec: int = 200000):
    x0 = _f64(x0)
    traj = np.zeros((maxrec, 5))
    ts = C.c_double(0)
    st = C.c_int32(0)
    n = lib().orc_trace_record(f.ref, C.byref(p), _dp(x0), _dp(traj), C.c_int64(maxrec),
                               C.byref(ts), C.byref(st))
    return traj[:n].copy(), ts.value, st.value


def trace_scripted(f: Field, p: CParams, x0, h):
    """Replays the step sizes h (1-D) from x0; returns xf, tstop, status, r[steps taken]."""
    x0, h = _f64(x0), _f64(h)
    xf = np.zeros(4)
    r = np.full(h.size, np.nan)
    ts = C.c_double(0)
    st = C.c_int32(0)
    n = lib().orc_trace_scripted(f.ref, C.byref(p), _dp(x0), C.c_int64(h.size), _dp(h), _dp(xf),
                                 C.byref(ts), C.byref(st), _dp(r))
    return xf, ts.value, st.value, r[:n].copy()


def tricubic_grad(f: Field, x, q: int = 0):
    """value and gradient (d/dx0, d/dx1, d/dx2) of quantity q's interpolant at x (reading R1c)"""
    v = C.c_double(0)
    g = np.zeros(3)
    lib().orc_tricubic_grad(f.ref, _dp(_f64(x)), C.c_int(q), C.byref(v), _dp(g))
    return v.value, g


def profile(f: Field, nodes, s: float):
    """value and d/ds of a profile tabulated on the unique s-nodes (the tables' piecewise cubic)"""
    v, d = C.c_double(0), C.c_double(0)
    nodes = _f64(nodes)
    lib().orc_profile(f.ref, _dp(nodes), C.c_double(s), C.byref(v), C.byref(d))
    return v.value, d.value


def hermite_state(y0, k0, y1, k1, h: float, theta: float) -> np.ndarray:
    """Cubic Hermite interpolant of a step's end states and end derivatives at theta in [0,1] (reading S5b)."""
    y = np.zeros(4)
    lib().orc_hermite_state(_dp(_f64(y0)), _dp(_f64(k0)), _dp(_f64(y1)), _dp(_f64(k1)), C.c_double(h),
                            C.c_double(theta), _dp(y))
    return y


def loss_refine(f: Field, y0, k0, y1, k1, h: float):
    """theta* in (0,1] and y(theta*): where the Hermite interpolant of the step crosses the loss boundary."""
    y = np.zeros(4)
    th = lib().orc_loss_refine(f.ref, _dp(_f64(y0)), _dp(_f64(k0)), _dp(_f64(y1)), _dp(_f64(k1)), C.c_double(h), _dp(y))
    return th, y


def estimate(g_kind, status=None, tstop=None, g_user=None):
    n = len(status) if status is not None else len(tstop if tstop is not None else g_user)
    out = np.zeros(3)
    st = np.ascontiguousarray(status, dtype=np.int32) if status is not None else None
    ts = _f64(tstop) if tstop is not None else None
    gu = _f64(g_user) if g_user is not None else None
    lib().orc_estimate(C.c_int(g_kind), C.c_int64(n),
                       st.ctypes.data_as(C.POINTER(C.c_int32)) if st is not None else None,
                       _dp(ts) if ts is not None else None, _dp(gu) if gu is not None else None,
                       _dp(out))
    return out


def lost_energy(f: Field, p: CParams, xf, mu, status) -> np.ndarray:
    """g_i = 1[lost] (vpar^2/2 + mu |B|(x_f)) / (v_total^2/2)  (reading G2)"""
    xf, mu = _f64(xf), _f64(mu)
    st = np.ascontiguousarray(status, dtype=np.int32)
    n = st.size
    g = np.zeros(n)
    lib().orc_lost_energy(f.ref, C.byref(p), C.c_int64(n), _dp(xf), _dp(mu), st.ctypes.data_as(C.POINTER(C.c_int32)),
                          _dp(g))
    return g


def exit_histogram(f: Field, xf, status, nb0: int, nb1: int) -> np.ndarray:
    """lost particles per bin of the exit point (reading G3): int64 [nb0][nb1]"""
    xf = _f64(xf)
    st = np.ascontiguousarray(status, dtype=np.int32)
    hist = np.zeros((nb0, nb1), dtype=np.int64)
    lib().orc_exit_histogram(f.ref, C.c_int64(st.size), _dp(xf), st.ctypes.data_as(C.POINTER(C.c_int32)),
                             C.c_int(nb0), C.c_int(nb1), hist.ctypes.data_as(C.POINTER(C.c_int64)))
    return hist


def max_threads() -> int:
    return int(lib().orc_max_threads())
