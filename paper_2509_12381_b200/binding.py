"""Thin ctypes binding of libaig.so (include/aig.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used here
for device memory and streams only.  There is no CPU fallback: if libaig.so is missing or
CUDA is unavailable the calls raise.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libaig.so")
_lib = None

EXPORTS = ["aig_workspace_bytes", "aig_integrate", "aig_histogram", "aig_step_once", "aig_run_host",
           "aig_fp64_peak_probe", "aig_kernel_info", "aig_kernel_launches", "aig_set_schedule", "aig_strerror",
           "aig_version", "aig_observables", "aig_outliers", "aig_outliers_workspace_bytes", "aig_trace",
           "aig_set_schedule_ex", "aig_get_schedule", "aig_map2d", "aig_outliers_static", "aig_outliers_static_max_n",
           "aig_potential"]


class AigError(RuntimeError):
    pass


class Params(C.Structure):
    _fields_ = [("m_ion", C.c_double), ("m_atom", C.c_double), ("C4", C.c_double), ("C8", C.c_double),
                ("a", C.c_double * 3), ("q", C.c_double * 3), ("omega_rf", C.c_double),
                ("t0", C.c_double), ("r_exit", C.c_double), ("r_turn", C.c_double),
                ("max_steps", C.c_int64), ("n_att", C.c_int32), ("n_rep", C.c_int32)]


class Out(C.Structure):
    _fields_ = [("y_final", C.c_void_p), ("t_final", C.c_void_p), ("lifetime", C.c_void_p),
                ("angle", C.c_void_p), ("r_min", C.c_void_p), ("n_acc", C.c_void_p),
                ("n_rej", C.c_void_p), ("n_turn", C.c_void_p), ("status", C.c_void_p),
                ("complex_flag", C.c_void_p), ("x_turn1", C.c_void_p)]   # x_turn1: optional, None = not recorded


class HistSpec(C.Structure):
    _fields_ = [("angle_edges", C.c_void_p), ("n_angle_bins", C.c_int32),
                ("life_edges", C.c_void_p), ("n_life_bins", C.c_int32), ("n_turn_bins", C.c_int32)]


class Hist(C.Structure):
    _fields_ = [("angle", C.c_void_p), ("lifetime", C.c_void_p), ("n_turn", C.c_void_p),
                ("status", C.c_void_p), ("totals", C.c_void_p)]


OUT_FIELDS = ("y_final", "t_final", "lifetime", "angle", "r_min", "n_acc", "n_rej", "n_turn", "status",
              "complex_flag")


def lib():
    """Load libaig.so (fails loudly when it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise AigError(f"{LIB_PATH} is missing: run `python -m paper_2509_12381_b200.build` "
                           "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.aig_workspace_bytes.restype = C.c_size_t
        L.aig_workspace_bytes.argtypes = [C.c_int64]
        L.aig_integrate.restype = C.c_int
        L.aig_integrate.argtypes = [C.POINTER(Params), C.c_void_p, C.c_int64, C.c_double, C.c_double,
                                    C.c_double, C.POINTER(Out), C.c_void_p, C.c_void_p]
        L.aig_histogram.restype = C.c_int
        L.aig_histogram.argtypes = [C.POINTER(Out), C.c_int64, C.POINTER(HistSpec), C.POINTER(Hist), C.c_void_p]
        L.aig_step_once.restype = C.c_int
        L.aig_step_once.argtypes = [C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64,
                                    C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.aig_run_host.restype = C.c_int
        L.aig_run_host.argtypes = [C.POINTER(Params), C.c_void_p, C.c_int64, C.c_double, C.c_double,
                                   C.c_double, C.POINTER(Out), C.POINTER(HistSpec), C.POINTER(Hist)]
        L.aig_fp64_peak_probe.restype = C.c_int
        L.aig_fp64_peak_probe.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.aig_kernel_info.restype = C.c_int
        L.aig_kernel_info.argtypes = [C.POINTER(C.c_int)] * 5
        L.aig_strerror.restype = C.c_char_p
        L.aig_strerror.argtypes = [C.c_int]
        L.aig_version.restype = C.c_int
        L.aig_kernel_launches.restype = C.c_uint64
        L.aig_kernel_launches.argtypes = []
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise AigError(f"{what} failed: {lib().aig_strerror(rc).decode()} (code {rc})")


def make_params(m_ion, m_atom, C4, C8, a, q, omega_rf, t0=0.0, r_exit=0.0, r_turn=math.inf,
                max_steps=1_000_000, n_att=0, n_rep=0) -> Params:
    """n_att, n_rep: exponents of V = -C_n/r^n + C_m/r^m with C_n = C4, C_m = C8 (0, 0 = the 4-8 benchmark potential)."""
    p = Params()
    p.n_att, p.n_rep = int(n_att), int(n_rep)
    p.m_ion, p.m_atom, p.C4, p.C8 = m_ion, m_atom, C4, C8
    for k in range(3):
        p.a[k] = a[k]
        p.q[k] = q[k]
    p.omega_rf, p.t0, p.r_exit, p.r_turn, p.max_steps = omega_rf, t0, r_exit, r_turn, int(max_steps)
    return p


POT_CNCM, POT_CNDE, POT_DERE = 0, 1, 2


def aig_potential(mode: int, n: int, m: int, a: float, b: float) -> dict:
    """The paper's potential front-end (include/aig.h: aig_potential): host arithmetic in the library.
    Returns {"Cn", "Cm", "De", "Re"}."""
    L = lib()
    L.aig_potential.restype = C.c_int
    L.aig_potential.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double] + [C.POINTER(C.c_double)] * 4
    v = [C.c_double() for _ in range(4)]
    _check(L.aig_potential(mode, n, m, a, b, *[C.byref(x) for x in v]), "aig_potential")
    return dict(zip(("Cn", "Cm", "De", "Re"), (x.value for x in v)))


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise AigError("CUDA device required: libaig has no CPU fallback")
    return torch


def _stream_ptr(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def alloc_out(N: int, device="cuda", position: bool = False):
    """Caller-owned device buffers for aig_integrate (dict of torch tensors).  position=True adds the
    optional x_turn1 [3, N] (ion position at the first bounce)."""
    torch = _torch()
    f8 = dict(dtype=torch.float64, device=device)
    i4 = dict(dtype=torch.int32, device=device)
    extra = dict(x_turn1=torch.empty((3, N), **f8)) if position else {}
    return dict(**extra, y_final=torch.empty((12, N), **f8), t_final=torch.empty(N, **f8),
                lifetime=torch.empty(N, **f8), angle=torch.empty(N, **f8), r_min=torch.empty(N, **f8),
                n_acc=torch.empty(N, **i4), n_rej=torch.empty(N, **i4), n_turn=torch.empty(N, **i4),
                status=torch.empty(N, **i4), complex_flag=torch.empty(N, dtype=torch.uint8, device=device))


def _out_struct(bufs) -> Out:
    o = Out()
    for f in OUT_FIELDS:
        setattr(o, f, bufs[f].data_ptr())
    o.x_turn1 = bufs["x_turn1"].data_ptr() if bufs.get("x_turn1") is not None else None
    return o


def workspace_bytes(N: int) -> int:
    return int(lib().aig_workspace_bytes(N))


def aig_integrate(params: Params, y0, t_max, rtol, atol, out=None, workspace=None, stream=None):
    """y0: CUDA float64 tensor [12, N] (contiguous).  Returns the dict of output tensors.
    Asynchronous on ``stream`` (default: torch's current stream)."""
    torch = _torch()
    assert y0.is_cuda and y0.dtype == torch.float64 and y0.dim() == 2 and y0.shape[0] == 12 and y0.is_contiguous()
    N = y0.shape[1]
    if out is None:
        out = alloc_out(N, y0.device)
    if workspace is None:
        workspace = torch.empty(workspace_bytes(N), dtype=torch.uint8, device=y0.device)
    o = _out_struct(out)
    rc = lib().aig_integrate(C.byref(params), y0.data_ptr(), N, t_max, rtol, atol, C.byref(o),
                             workspace.data_ptr(), _stream_ptr(stream))
    _check(rc, "aig_integrate")
    out["_workspace"] = workspace  # keep alive until the stream has run
    return out


def alloc_hist(n_angle: int, n_life: int, n_turn_bins: int = 64, device="cuda"):
    torch = _torch()
    z = lambda n: torch.zeros(n, dtype=torch.int64, device=device)  # uint64 bit pattern
    return dict(angle=z(n_angle + 2), lifetime=z(n_life + 2), n_turn=z(n_turn_bins), status=z(4), totals=z(4))


def aig_histogram(obs, angle_edges, life_edges, n_turn_bins: int = 64, hist=None, stream=None):
    """obs: dict from aig_integrate; edges: CUDA float64 tensors (strictly increasing).
    Accumulates into ``hist`` (allocated zeroed when None)."""
    torch = _torch()
    for e in (angle_edges, life_edges):
        assert e.is_cuda and e.dtype == torch.float64 and e.is_contiguous() and e.numel() >= 2
    na, nl = angle_edges.numel() - 1, life_edges.numel() - 1
    N = obs["angle"].numel()
    if hist is None:
        hist = alloc_hist(na, nl, n_turn_bins, obs["angle"].device)
    spec = HistSpec(angle_edges.data_ptr(), na, life_edges.data_ptr(), nl, n_turn_bins)
    h = Hist(*[hist[k].data_ptr() for k in ("angle", "lifetime", "n_turn", "status", "totals")])
    o = _out_struct(obs)
    rc = lib().aig_histogram(C.byref(o), N, C.byref(spec), C.byref(h), _stream_ptr(stream))
    _check(rc, "aig_histogram")
    return hist


class ObsExtra(C.Structure):
    _fields_ = [("dist", C.c_void_p), ("KE", C.c_void_p), ("transfer", C.c_void_p), ("position", C.c_void_p)]


# order of aig_outliers' result rows
OUTLIER_KEYS = ("angle", "n_turn", "lifetime", "transfer", "dist", "n_acc", "KE", "position")


def _extra_struct(extra) -> ObsExtra:
    pos = extra.get("position")
    return ObsExtra(extra["dist"].data_ptr(), extra["KE"].data_ptr(), extra["transfer"].data_ptr(),
                    pos.data_ptr() if pos is not None else None)


def aig_observables(params: Params, y0, obs, extra=None, stream=None):
    """dist, KE, transfer (include/aig.h) of the trajectories in ``obs`` (dict from aig_integrate), and
    position when ``obs`` holds x_turn1 (alloc_out(position=True))."""
    torch = _torch()
    N = y0.shape[1]
    assert y0.is_cuda and y0.dtype == torch.float64 and y0.shape[0] == 12 and y0.is_contiguous()
    if extra is None:
        keys = ("dist", "KE", "transfer") + (("position",) if obs.get("x_turn1") is not None else ())
        extra = {k: torch.empty(N, dtype=torch.float64, device=y0.device) for k in keys}
    e = _extra_struct(extra)
    o = _out_struct(obs)
    L = lib()
    L.aig_observables.restype = C.c_int
    L.aig_observables.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    _check(L.aig_observables(C.byref(params), y0.data_ptr(), C.byref(o), N, C.byref(e), _stream_ptr(stream)),
           "aig_observables")
    return extra


def aig_outliers(obs, extra, stream=None):
    """int64 CUDA tensor [8, 2]: index of the smallest / largest value of each OUTLIER_KEYS observable
    (row "position" is -1, -1 when ``extra`` has none)."""
    torch = _torch()
    N = obs["angle"].numel()
    dev = obs["angle"].device
    L = lib()
    L.aig_outliers_workspace_bytes.restype = C.c_size_t
    L.aig_outliers.restype = C.c_int
    L.aig_outliers.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
    ws = torch.empty(int(L.aig_outliers_workspace_bytes()), dtype=torch.uint8, device=dev)
    res = torch.empty((len(OUTLIER_KEYS), 2), dtype=torch.int64, device=dev)
    e = _extra_struct(extra)
    o = _out_struct(obs)
    _check(L.aig_outliers(C.byref(o), C.byref(e), N, res.data_ptr(), ws.data_ptr(), _stream_ptr(stream)), "aig_outliers")
    res._ws = ws  # keep the scratch alive until the stream has run
    return res


def aig_outliers_static(obs, extra, result, stream=None):
    """aig_outliers through the library's built-in scratch (include/aig.h): nothing is allocated here or in the
    library, so the caller passes ``result``, an int64 CUDA tensor [8, 2] of its own, and gets it back.  For callers
    that hold their arrays already and may not ask for more device memory.  Calls on one device must not overlap
    (one shared scratch); raises for N beyond aig_outliers_static_max_n()."""
    torch = _torch()
    N = obs["angle"].numel()
    assert result.is_cuda and result.dtype == torch.int64 and tuple(result.shape) == (len(OUTLIER_KEYS), 2)
    assert result.is_contiguous()
    L = lib()
    L.aig_outliers_static.restype = C.c_int
    L.aig_outliers_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    e = _extra_struct(extra)
    o = _out_struct(obs)
    _check(L.aig_outliers_static(C.byref(o), C.byref(e), N, result.data_ptr(), _stream_ptr(stream)),
           "aig_outliers_static")
    return result


def aig_outliers_static_max_n() -> int:
    L = lib()
    L.aig_outliers_static_max_n.restype = C.c_int64
    return int(L.aig_outliers_static_max_n())


class MapSpec(C.Structure):
    _fields_ = [("u_edges", C.c_void_p), ("n_u", C.c_int32), ("phi_edges", C.c_void_p), ("n_phi", C.c_int32)]


def aig_map2d(y0, value, u_edges, phi_edges, count=None, total=None, stream=None):
    """An observable against the launch direction (include/aig.h: aig_map2d): returns (count [n_u, n_phi] int64,
    sum [n_u, n_phi] float64) CUDA tensors, accumulated into when given."""
    torch = _torch()
    N = y0.shape[1]
    assert y0.is_cuda and y0.dtype == torch.float64 and y0.shape[0] == 12 and y0.is_contiguous()
    assert value.is_cuda and value.dtype == torch.float64 and value.numel() == N and value.is_contiguous()
    for e in (u_edges, phi_edges):
        assert e.is_cuda and e.dtype == torch.float64 and e.is_contiguous() and e.numel() >= 2
    nu, nph = u_edges.numel() - 1, phi_edges.numel() - 1
    if count is None:
        count = torch.zeros((nu, nph), dtype=torch.int64, device=y0.device)
    if total is None:
        total = torch.zeros((nu, nph), dtype=torch.float64, device=y0.device)
    spec = MapSpec(u_edges.data_ptr(), nu, phi_edges.data_ptr(), nph)
    L = lib()
    L.aig_map2d.restype = C.c_int
    L.aig_map2d.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    _check(L.aig_map2d(y0.data_ptr(), N, value.data_ptr(), C.byref(spec), count.data_ptr(), total.data_ptr(),
                       _stream_ptr(stream)), "aig_map2d")
    return count, total


def aig_trace(params: Params, y0, t_max, rtol, atol, cap: int = 1 << 20, stream=None):
    """Replay one trajectory (y0: CUDA float64 [12]); returns (t [cap], y [12, cap], n [4]) CUDA tensors,
    n = (accepted steps, status, failed attempts, turning points); rows beyond min(n[0], cap) are unset."""
    torch = _torch()
    assert y0.is_cuda and y0.dtype == torch.float64 and y0.numel() == 12 and y0.is_contiguous()
    t = torch.empty(cap, dtype=torch.float64, device=y0.device)
    y = torch.empty((12, cap), dtype=torch.float64, device=y0.device)
    n = torch.zeros(4, dtype=torch.int64, device=y0.device)
    L = lib()
    L.aig_trace.restype = C.c_int
    L.aig_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_int64, C.c_void_p,
                            C.c_void_p, C.c_void_p, C.c_void_p]
    _check(L.aig_trace(C.byref(params), y0.data_ptr(), t_max, rtol, atol, cap, t.data_ptr(), y.data_ptr(),
                       n.data_ptr(), _stream_ptr(stream)), "aig_trace")
    return t, y, n


def aig_step_once(params: Params, y, t, h, rtol, atol, stream=None):
    torch = _torch()
    assert y.is_cuda and y.dtype == torch.float64 and y.shape[0] == 12 and y.is_contiguous()
    N = y.shape[1]
    ynew = torch.empty_like(y)
    err = torch.empty(N, dtype=torch.float64, device=y.device)
    rc = lib().aig_step_once(C.byref(params), y.data_ptr(), t.data_ptr(), h.data_ptr(), N, rtol, atol,
                             ynew.data_ptr(), err.data_ptr(), _stream_ptr(stream))
    _check(rc, "aig_step_once")
    return ynew, err


def aig_run_host(params: Params, y0_host: np.ndarray, t_max, rtol, atol, angle_edges=None, life_edges=None,
                 n_turn_bins: int = 64, want=OUT_FIELDS, out=None):
    """End-to-end call on HOST numpy buffers (H2D + kernels + D2H inside, blocking).
    ``want`` selects which per-trajectory outputs are copied back."""
    y0_host = np.ascontiguousarray(y0_host, dtype=np.float64)
    N = y0_host.shape[1]
    dt = dict(y_final=(np.float64, (12, N)), t_final=(np.float64, (N,)), lifetime=(np.float64, (N,)),
              angle=(np.float64, (N,)), r_min=(np.float64, (N,)), n_acc=(np.int32, (N,)),
              n_rej=(np.int32, (N,)), n_turn=(np.int32, (N,)), status=(np.int32, (N,)),
              complex_flag=(np.uint8, (N,)), x_turn1=(np.float64, (3, N)))
    res = {} if out is None else out
    o = Out()
    for f in OUT_FIELDS + ("x_turn1",):
        if f in want:
            if f not in res:
                res[f] = np.empty(dt[f][1], dtype=dt[f][0])
            setattr(o, f, res[f].ctypes.data)
        else:
            setattr(o, f, None)
    spec_p, hist_p = None, None
    if angle_edges is not None:
        ae = np.ascontiguousarray(angle_edges, dtype=np.float64)
        le = np.ascontiguousarray(life_edges, dtype=np.float64)
        hist = dict(angle=np.zeros(len(ae) + 1, np.uint64), lifetime=np.zeros(len(le) + 1, np.uint64),
                    n_turn=np.zeros(n_turn_bins, np.uint64), status=np.zeros(4, np.uint64),
                    totals=np.zeros(4, np.uint64))
        spec = HistSpec(ae.ctypes.data, len(ae) - 1, le.ctypes.data, len(le) - 1, n_turn_bins)
        h = Hist(*[hist[k].ctypes.data for k in ("angle", "lifetime", "n_turn", "status", "totals")])
        spec_p, hist_p = C.byref(spec), C.byref(h)
        res["hist"] = hist
    rc = lib().aig_run_host(C.byref(params), y0_host.ctypes.data, N, t_max, rtol, atol, C.byref(o), spec_p, hist_p)
    _check(rc, "aig_run_host")
    return res


def fp64_peak_probe(iters: int = 4096, ilp: int = 8):
    f, ms = C.c_double(0), C.c_double(0)
    _check(lib().aig_fp64_peak_probe(iters, ilp, C.byref(f), C.byref(ms)), "aig_fp64_peak_probe")
    return f.value, ms.value


def kernel_info() -> dict:
    v = [C.c_int(0) for _ in range(5)]
    _check(lib().aig_kernel_info(*[C.byref(x) for x in v]), "aig_kernel_info")
    keys = ("sm_count", "blocks_per_sm", "threads_per_block", "regs_per_thread", "local_bytes_per_thread")
    return dict(zip(keys, [x.value for x in v]))


class Schedule(C.Structure):
    """include/aig.h: aig_schedule."""
    _fields_ = [("tail_iters", C.c_int32), ("budget", C.c_int32), ("split_sms", C.c_int32), ("split_grid", C.c_int32),
                ("plan", C.c_int32), ("kappa", C.c_double), ("depth", C.c_int32), ("mean_factor", C.c_int32),
                ("drain_lanes", C.c_int32), ("slow0", C.c_double), ("slow1", C.c_double),
                ("refill_batch", C.c_int32), ("refill_wait", C.c_int32), ("poll_iters", C.c_int32),
                ("hist_blocks_per_sm", C.c_int32)]


def get_schedule() -> dict:
    s = Schedule()
    L = lib()
    L.aig_get_schedule.restype = C.c_int
    _check(L.aig_get_schedule(C.byref(s)), "aig_get_schedule")
    return {k: getattr(s, k) for k, _ in Schedule._fields_}


def set_schedule(**knobs) -> None:
    """Test / tuning hook (include/aig.h: aig_set_schedule_ex); never changes a result.  The library's
    defaults with the given knobs replaced; no argument = the defaults."""
    L = lib()
    L.aig_set_schedule_ex.restype = C.c_int
    L.aig_set_schedule_ex.argtypes = [C.c_void_p]
    cur = get_schedule()
    _check(L.aig_set_schedule_ex(None), "aig_set_schedule_ex")
    if not knobs:
        return
    s = Schedule(**get_schedule())
    for k, v in knobs.items():
        if k not in dict(Schedule._fields_):
            raise TypeError(f"unknown schedule knob {k!r}")
        setattr(s, k, v)
    rc = L.aig_set_schedule_ex(C.cast(C.byref(s), C.c_void_p))
    if rc:
        L.aig_set_schedule_ex(C.cast(C.byref(Schedule(**cur)), C.c_void_p))  # leave the schedule as it was
    _check(rc, "aig_set_schedule_ex")


def kernel_launches() -> int:
    """Kernels libaig has launched in this process so far."""
    return int(lib().aig_kernel_launches())


def hist_to_numpy(hist) -> dict:
    """Device histogram dict -> numpy uint64 arrays (synchronises)."""
    return {k: v.cpu().numpy().view(np.uint64) for k, v in hist.items()}
