"""aig_outliers_static: the outliers pass for callers that cannot allocate device memory.

Who that is: code that runs inside somebody else's memory plan -- an analysis step called between batches of a long
ensemble run whose driver program gave away all of the GPU's memory at start-up and forbids cudaMalloc afterwards
(a late allocation stalls every stream of the device and may simply fail), or a plug-in of a framework that owns the
allocator.  Such a caller has its observable arrays and a result buffer, but nothing to hand aig_outliers as a
workspace.  aig_outliers_static keeps that scratch in a fixed array inside libaig (include/aig.h), shared by all
calls on a device and never cleared between them.

What is checked: the indices it returns equal those of aig_outliers (the existing path, itself checked against the
oracle in test_gpu_parity.py) exactly -- this is integer work, the tolerance of the outliers tests is zero -- on two
calls in a row, the second on fewer trajectories with NaNs and ties, so that what the first call left in the shared
scratch (partials of blocks the second launch does not have, a used ticket counter) would show if it were read.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It makes no assumption about what ran before it in the process (the look-up of the scratch address
happens at the first call on the device, whenever that is).
"""
import ctypes as C

import numpy as np
import pytest

from paper_2509_12381_b200 import inputs


def test_static_limit_is_refused_on_the_host():
    """N beyond the stated maximum: a named error before anything touches the device (no GPU needed)."""
    from paper_2509_12381_b200 import binding, build as aig_build
    aig_build.build()
    L = binding.lib()
    L.aig_outliers_static.restype = C.c_int
    L.aig_outliers_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    nmax = binding.aig_outliers_static_max_n()
    assert nmax == 1 << 28
    fake_result = C.c_void_p(4096)            # aligned, never dereferenced: the size check comes first
    rc = L.aig_outliers_static(None, None, nmax + 1, fake_result, None)
    assert rc == -8
    L.aig_strerror.restype = C.c_char_p
    msg = L.aig_strerror(rc)
    assert b"AIG_OUTLIERS_STATIC_MAX_N" in msg and b"aig_outliers" in msg
    assert L.aig_outliers_static(None, None, -1, fake_result, None) == -2
    assert L.aig_outliers_static(None, None, 10, None, None) == -1
    assert L.aig_outliers_static(None, None, 10, fake_result, None) == -1     # N > 0 needs the arrays


@pytest.mark.gpu
def test_outliers_static_matches_outliers_twice_in_a_row():
    import torch
    from paper_2509_12381_b200 import binding as aig
    aig.lib()
    assert torch.cuda.is_available()
    dev = torch.device("cuda")
    # call 1: real observables of a small ensemble (several blocks and a ragged tail; a quarter without a bounce,
    # so `position` holds NaNs)
    w = inputs.config(2).replace(N=20000 + 13, r_turn=3000.0)
    y0 = torch.from_numpy(np.ascontiguousarray(inputs.generate_y0(w))).cuda()
    p = aig.make_params(**w.params())
    out = aig.aig_integrate(p, y0, w.t_max, w.rtol, w.atol, out=aig.alloc_out(w.N, "cuda", position=True))
    extra = aig.aig_observables(p, y0, out)
    want1 = aig.aig_outliers(out, extra).cpu().numpy()
    res = torch.full((8, 2), -7, dtype=torch.int64, device=dev)     # the caller's buffer, reused by both calls
    got1 = aig.aig_outliers_static(out, extra, res).cpu().numpy()
    assert np.array_equal(got1, want1), (got1, want1)
    assert (want1[:7] >= 0).all()
    # call 2, straight after: the first 1000 trajectories only (4 blocks instead of 79), with NaNs and ties
    n2 = 1000
    out2 = {k: v[..., :n2].clone() for k, v in out.items() if not k.startswith("_")}    # copies: `out` is used again below
    extra2 = {k: v[:n2].clone() for k, v in extra.items()}
    out2["lifetime"][::3] = float("nan")
    out2["angle"][:] = 1.0
    want2 = aig.aig_outliers(out2, extra2).cpu().numpy()
    got2 = aig.aig_outliers_static(out2, extra2, res).cpu().numpy()
    assert np.array_equal(got2, want2), (got2, want2)
    assert tuple(got2[0]) == (0, 0) and got2.max() < n2
    assert not np.array_equal(got1, got2)
    # and the first input once more: nothing of call 2 sticks either
    assert np.array_equal(aig.aig_outliers_static(out, extra, res).cpu().numpy(), want1)
    # N = 0: every row -1
    empty = aig.alloc_out(0, dev)
    ex0 = {k: torch.empty(0, dtype=torch.float64, device=dev) for k in ("dist", "KE", "transfer")}
    assert np.all(aig.aig_outliers_static(empty, ex0, res).cpu().numpy() == -1)
    # beyond the stated maximum: refused by name (the binding raises with the library's message)
    L = aig.lib()
    L.aig_outliers_static.restype = C.c_int
    L.aig_outliers_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    assert L.aig_outliers_static(None, None, aig.aig_outliers_static_max_n() + 1, res.data_ptr(), None) == -8
