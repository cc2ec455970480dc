"""ctypes front-end of the CPU oracle (oracle/aig_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from the
product package and the product imports nothing from here.

The histogram oracle is the plain definition written with ``numpy.searchsorted``
(SURVEY.md 8(c) O6 "Histogram"); everything else calls the C file, which is compiled
here with ``gcc -O2 -ffp-contract=off`` (no FMA contraction: one IEEE operation per
operator, in source order).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "aig_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None


class OrcParams(C.Structure):
    _fields_ = [("m_ion", C.c_double), ("m_atom", C.c_double), ("C4", C.c_double), ("C8", C.c_double),
                ("a", C.c_double * 3), ("q", C.c_double * 3), ("omega_rf", C.c_double),
                ("t0", C.c_double), ("r_exit", C.c_double), ("r_turn", C.c_double),
                ("max_steps", C.c_int64), ("n_att", C.c_int32), ("n_rep", C.c_int32)]


RHS_FN = C.CFUNCTYPE(None, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int, C.c_void_p)
OBS_FN = C.CFUNCTYPE(C.c_int, C.c_double, C.POINTER(C.c_double), C.c_void_p)


def build(force: bool = False) -> str:
    """Compile liboracle.so (idempotent).  Building the checker is not using it."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c11",
                                   "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_dp45_step.restype = C.c_int
        _lib.orc_dp45_integrate.restype = C.c_int
        _lib.orc_integrate.restype = C.c_int
        _lib.orc_integrate_trace.restype = C.c_int
        _lib.orc_step_once.restype = C.c_int
        _lib.orc_rhs_batch.restype = C.c_int
    return _lib


def make_params(m_ion, m_atom, C4, C8, a, q, omega_rf, t0=0.0, r_exit=0.0, r_turn=float("inf"),
                max_steps=1_000_000, n_att=0, n_rep=0) -> OrcParams:
    """n_att, n_rep: exponents of V = -C_n/r^n + C_m/r^m with C_n = C4, C_m = C8 (0, 0 = the 4-8 benchmark potential)."""
    p = OrcParams()
    p.n_att, p.n_rep = int(n_att), int(n_rep)
    p.m_ion, p.m_atom, p.C4, p.C8 = m_ion, m_atom, C4, C8
    for k in range(3):
        p.a[k] = a[k]
        p.q[k] = q[k]
    p.omega_rf, p.t0, p.r_exit, p.r_turn, p.max_steps = omega_rf, t0, r_exit, r_turn, int(max_steps)
    return p


def _dp(x):
    return x.ctypes.data_as(C.POINTER(C.c_double))


def _ip(x):
    return x.ctypes.data_as(C.POINTER(C.c_int32))


def tableau():
    """(c[7], A[7][6], E[7]) exactly as the C code holds them."""
    c = np.zeros(7)
    a = np.zeros((7, 6))
    e = np.zeros(7)
    lib().orc_tableau(_dp(c), _dp(a), _dp(e))
    return c, a, e


def rhs(p: OrcParams, t, y):
    """f(t_i, y[:, i]) for every column of y[12][N]."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    N = y.shape[1]
    t = np.ascontiguousarray(np.broadcast_to(np.asarray(t, dtype=np.float64), (N,)))
    f = np.empty_like(y)
    rc = lib().orc_rhs_batch(C.byref(p), _dp(t), _dp(y), C.c_int64(N), _dp(f))
    assert rc == 0
    return f


def step_once(p: OrcParams, y, t, h, rtol, atol):
    """One attempted DP5(4) step per column: returns (ynew[12][N], err[N])."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    N = y.shape[1]
    t = np.ascontiguousarray(np.broadcast_to(np.asarray(t, dtype=np.float64), (N,)))
    h = np.ascontiguousarray(np.broadcast_to(np.asarray(h, dtype=np.float64), (N,)))
    ynew = np.empty_like(y)
    err = np.empty(N)
    rc = lib().orc_step_once(C.byref(p), _dp(y), _dp(t), _dp(h), C.c_int64(N), C.c_double(rtol),
                             C.c_double(atol), _dp(ynew), _dp(err))
    if rc:
        raise ValueError(f"orc_step_once rc={rc}")
    return ynew, err


def integrate(p: OrcParams, y0, t_max, rtol, atol, threads: int = 1) -> dict:
    """Integrate every column of y0[12][N].  ``threads`` > 1 only splits the index range
    over Python threads (ctypes releases the GIL); each trajectory is still computed by the
    same single-threaded code, so results do not depend on ``threads``."""
    y0 = np.ascontiguousarray(y0, dtype=np.float64)
    assert y0.ndim == 2 and y0.shape[0] == 12
    N = y0.shape[1]
    out = dict(y_final=np.zeros((12, N)), t_final=np.zeros(N), lifetime=np.zeros(N), angle=np.zeros(N),
               r_min=np.zeros(N), n_acc=np.zeros(N, np.int32), n_rej=np.zeros(N, np.int32),
               n_turn=np.zeros(N, np.int32), status=np.zeros(N, np.int32),
               complex_flag=np.zeros(N, np.uint8), x_turn1=np.zeros((3, N)))
    L = lib()

    def run(lo, hi):
        rc = L.orc_integrate(C.byref(p), _dp(y0), C.c_int64(N), C.c_double(t_max), C.c_double(rtol),
                             C.c_double(atol), C.c_int64(lo), C.c_int64(hi), _dp(out["y_final"]),
                             _dp(out["t_final"]), _dp(out["lifetime"]), _dp(out["angle"]),
                             _dp(out["r_min"]), _ip(out["n_acc"]), _ip(out["n_rej"]),
                             _ip(out["n_turn"]), _ip(out["status"]),
                             out["complex_flag"].ctypes.data_as(C.POINTER(C.c_uint8)), _dp(out["x_turn1"]))
        if rc:
            raise ValueError(f"orc_integrate rc={rc}")

    threads = max(1, min(int(threads), N if N else 1))
    if threads == 1:
        run(0, N)
    else:
        # interleave small chunks so long trajectories spread over the threads
        chunk = max(1, min(256, N // (threads * 8) or 1))
        bounds = [(lo, min(N, lo + chunk)) for lo in range(0, N, chunk)]
        it = iter(bounds)
        errs = []

        def worker():
            try:
                while True:
                    with _lock:
                        b = next(it, None)
                    if b is None:
                        return
                    run(*b)
            except Exception as e:  # pragma: no cover
                errs.append(e)

        ts = [threading.Thread(target=worker) for _ in range(threads)]
        [t.start() for t in ts]
        [t.join() for t in ts]
        if errs:
            raise errs[0]
    return out


def integrate_trace(p: OrcParams, y0, t_max, rtol, atol, cap: int = 200000):
    """One trajectory with every accepted step recorded: (t[n], y[n][12], status)."""
    y0 = np.ascontiguousarray(y0, dtype=np.float64).reshape(12)
    tt = np.zeros(cap)
    yy = np.zeros((cap, 12))
    n = C.c_int64(0)
    st = C.c_int(0)
    rc = lib().orc_integrate_trace(C.byref(p), _dp(y0), C.c_double(t_max), C.c_double(rtol),
                                   C.c_double(atol), _dp(tt), _dp(yy), C.c_int64(cap), C.byref(n),
                                   C.byref(st))
    if rc:
        raise ValueError(f"orc_integrate_trace rc={rc}")
    return tt[:n.value].copy(), yy[:n.value].copy(), st.value


# ---- generic right-hand sides through the SAME stepper (pins on y'=-y etc.) -----------------

def _wrap_rhs(fun, n):
    def cb(t, yp, fp, nn, _ctx):
        y = np.ctypeslib.as_array(yp, shape=(n,))
        f = np.ctypeslib.as_array(fp, shape=(n,))
        f[:] = fun(t, y)
    return RHS_FN(cb)


def generic_step(fun, t, y, h, rtol=1e-6, atol=1e-9):
    """One attempted step of the oracle's stepper on y' = fun(t, y): (ynew, err)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    n = y.size
    cb = _wrap_rhs(fun, n)
    ynew = np.zeros(n)
    err = C.c_double(0)
    rc = lib().orc_dp45_step(cb, None, C.c_int(n), C.c_double(t), _dp(y), C.c_double(h),
                             C.c_double(rtol), C.c_double(atol), _dp(ynew), C.byref(err))
    if rc:
        raise ValueError(f"orc_dp45_step rc={rc}")
    return ynew, err.value


def generic_integrate(fun, t0, y0, t_max, rtol, atol, max_steps=1_000_000, observe=None, cap=0):
    """The oracle's adaptive loop on y' = fun(t, y).  Returns dict(t, y, n_acc, n_rej, status
    [, trace_t, trace_y])."""
    y0 = np.ascontiguousarray(y0, dtype=np.float64)
    n = y0.size
    cb = _wrap_rhs(fun, n)
    ocb = None
    if observe is not None:
        def _o(t, yp, _ctx):
            return int(bool(observe(t, np.ctypeslib.as_array(yp, shape=(n,)))))
        ocb = OBS_FN(_o)
    yf = np.zeros(n)
    tf = C.c_double(0)
    na, nr, ntr = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    st = C.c_int(0)
    tt = np.zeros(max(cap, 1))
    yy = np.zeros((max(cap, 1), n))
    rc = lib().orc_dp45_integrate(cb, None, C.c_int(n), C.c_double(t0), _dp(y0), C.c_double(t_max),
                                  C.c_double(rtol), C.c_double(atol), C.c_int64(max_steps),
                                  ocb if ocb is not None else C.cast(None, OBS_FN), None, _dp(yf),
                                  C.byref(tf), C.byref(na), C.byref(nr), C.byref(st),
                                  _dp(tt) if cap else None, _dp(yy) if cap else None,
                                  C.c_int64(cap), C.byref(ntr))
    if rc:
        raise ValueError(f"orc_dp45_integrate rc={rc}")
    res = dict(t=tf.value, y=yf, n_acc=na.value, n_rej=nr.value, status=st.value)
    if cap:
        res["trace_t"] = tt[:ntr.value].copy()
        res["trace_y"] = yy[:ntr.value].copy()
    return res


# ---- histogram oracle: the plain definition ---------------------------------------------------

def _bin_counts(v, edges):
    """counts[0] = underflow (v < edges[0]); counts[1+j] = edges[j] <= v < edges[j+1];
    counts[nb+1] = overflow (v >= edges[nb], and NaN)."""
    v = np.asarray(v, dtype=np.float64)
    nb = len(edges) - 1
    j = np.searchsorted(edges, v, side="right")  # number of edges <= v ; NaN sorts last -> nb+1
    return np.bincount(j, minlength=nb + 2).astype(np.uint64)


def histogram(obs: dict, angle_edges, life_edges, n_turn_bins: int = 64) -> dict:
    """Device-side observable reduction, as a definition."""
    cf = np.asarray(obs["complex_flag"]).astype(bool)
    nt = np.minimum(np.asarray(obs["n_turn"]).astype(np.int64), n_turn_bins - 1)
    st = np.asarray(obs["status"]).astype(np.int64)
    N = len(st)
    return dict(
        angle=_bin_counts(obs["angle"], np.asarray(angle_edges)),
        lifetime=_bin_counts(np.asarray(obs["lifetime"])[cf], np.asarray(life_edges)),
        n_turn=np.bincount(nt, minlength=n_turn_bins).astype(np.uint64),
        status=np.bincount(st, minlength=4)[:4].astype(np.uint64),
        totals=np.array([np.asarray(obs["n_acc"]).astype(np.int64).sum(),
                         np.asarray(obs["n_rej"]).astype(np.int64).sum(),
                         int(cf.sum()), N], dtype=np.uint64),
    )


# ---------------------------------------------------------------------------------------------
# NEXT-1: the paper's remaining per-trajectory observables and its "outliers"
# ---------------------------------------------------------------------------------------------
OUTLIER_KEYS = ("angle", "n_turn", "lifetime", "transfer", "dist", "n_acc", "KE", "position")


def observables(p: OrcParams, y0, y_final, x_turn1=None) -> dict:
    """The observables of PAPER.md:495-497 that follow from the initial and final states alone,
    written as their definitions (float64, one trajectory per column):
      dist     final atom-ion distance                     |x_atom - x_ion| at the end
      KE       final kinetic energy of the ion             m_ion |v_ion|^2 / 2
      transfer momentum transferred by the atom            m_atom |v_atom(end) - v_atom(t0)|
      position how far the ion is from the origin during   |x_ion| at the step end that counts the first
               the first bounce (needs x_turn1[3][N] of     bounce; NaN for a trajectory without one
               integrate())
    (the paper names them without formulas; readings S24-S26 and S29 of DESIGN.md)."""
    y0 = np.asarray(y0, dtype=np.float64)
    yf = np.asarray(y_final, dtype=np.float64)
    d = yf[6:9] - yf[0:3]
    dv = yf[9:12] - y0[9:12]
    obs = {"dist": np.sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]),
           "KE": 0.5 * p.m_ion * (yf[3] * yf[3] + yf[4] * yf[4] + yf[5] * yf[5]),
           "transfer": p.m_atom * np.sqrt(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2])}
    if x_turn1 is not None:
        x = np.asarray(x_turn1, dtype=np.float64)
        obs["position"] = np.sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2])
    return obs


def outliers(obs: dict) -> dict:
    """PAPER.md:521 ("outliers.txt stores the initial conditions for the trajectories with the highest
    and lowest value of each observable"): for each observable of OUTLIER_KEYS the index of its
    smallest and of its largest value; the first index wins a tie; NaNs are skipped (an observable
    that is NaN everywhere, or N = 0, gives -1).  Plain loops over the definition."""
    out = {}
    for k in OUTLIER_KEYS:
        v = np.asarray(obs[k])
        lo = hi = -1
        for i in range(v.shape[0]):
            x = v[i]
            if x != x:
                continue
            if lo < 0 or x < v[lo]:
                lo = i
            if hi < 0 or x > v[hi]:
                hi = i
        out[k] = (lo, hi)
    return out


def map2d(y0, value, u_edges, phi_edges):
    """PAPER.md:483, :517 (an observable "as a function of the spherical angles theta and phi", the "(theta, phi) for
    the initial conditions of the atom"), as a definition: the direction of trajectory i is that of the ATOM's
    position at t0 (rows 6-8 alone, about the trap centre; the ion's thermal displacement does not enter);
    u = (1 - cos theta)/2, phi = atan2(y, x) brought into [phi_edges[0], phi_edges[0] + 2 pi) (a window may straddle
    phi = 0; at a pole x = y = 0 and phi = atan2(0, 0) = 0); cell (a, b) holds u_edges[a] <= u < u_edges[a+1],
    phi_edges[b] <= phi < phi_edges[b+1].  Returns (count, sum) of the non-NaN values inside the window,
    [n_u][n_phi].  Plain loop."""
    y0 = np.asarray(y0, dtype=np.float64)
    ue, pe = np.asarray(u_edges, dtype=np.float64), np.asarray(phi_edges, dtype=np.float64)
    nu, nph = len(ue) - 1, len(pe) - 1
    count = np.zeros((nu, nph), dtype=np.int64)
    total = np.zeros((nu, nph), dtype=np.float64)
    d = y0[6:9]
    r = np.sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2])
    with np.errstate(invalid="ignore", divide="ignore"):
        u = 0.5 * (1.0 - d[2] / r)
    phi = np.arctan2(d[1], d[0])
    two_pi = 2.0 * np.pi
    phi = phi - two_pi * np.floor((phi - pe[0]) / two_pi)
    a = np.searchsorted(ue, u, side="right")
    b = np.searchsorted(pe, phi, side="right")
    for i in range(y0.shape[1]):
        v = value[i]
        if 1 <= a[i] <= nu and 1 <= b[i] <= nph and v == v:
            count[a[i] - 1, b[i] - 1] += 1
            total[a[i] - 1, b[i] - 1] += v
    return count, total
