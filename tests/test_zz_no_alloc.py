"""fe_omega_grid_static: the one entry point of libfe that allocates nothing (include/fe.h has the contract).

Why it exists.  Every other call works on an fe_handle, and a handle allocates: fe_create makes the math tables, and
fe_omega_grid re-makes the handle's scratch with cudaFree + cudaMalloc whenever a call needs more than an earlier one did.
Some users of this library cannot have that: a job in which PyTorch's caching allocator (or anything else) already holds
nearly all of HBM, so that a cudaMalloc from outside that pool fails; a caller that runs other streams on the same GPU and
cannot afford the device-wide wait cudaMalloc / cudaFree cause; a service whose device-memory budget is fixed at start-up.
fe_omega_grid_static serves them on small grids: no handle, all working memory in one fixed array built into libfe.so.

What is checked here: its Omega against the existing path (fe_omega_grid: the default kernel, and the same direct
formulation, on the same inputs) within the 1e-12 the parity tests use, on two calls in a row, with a larger call in
between whose leftovers the second one must not pick up; and that sizes beyond the fixed limits are refused with a message
that says which limit.  This file is named so that pytest collects it last: it must pass both alone in a fresh process
(where its first call is also the first CUDA work of the process and does the one-time set-up) and after all other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1412_8754_b200 import workloads as W

pytestmark = pytest.mark.gpu

RTOL = 1e-12      # the Omega bar of tests/test_fe_gpu.py


def handle_path(fe, w, T, mode=None):
    import torch
    with fe.FreeEnergy(w.params, w.N, T) as F:
        if mode is not None:
            F.set_eval_mode(mode)
        om = F.omega_grid(w.q, w.h, w.delta)
        torch.cuda.synchronize()
        return om.cpu().numpy()


def max_rel(a, b):
    return float(np.max(np.abs(a - b) / np.maximum(np.abs(b), 1e-300)))


def test_static_entry_point_matches_existing_path_on_two_calls_in_a_row(fe):
    import torch
    small = W.ragged(seed=11, N=45, nq=3, nh=5, nd=37)                 # off-grid q, ragged tiles, negative h and Delta
    big = W.interior_minimum(N=256, U=5.0, T=0.004, nq=2, nh=24, nd=160)   # more k-chunks, more outputs: fills more scratch
    out_small = torch.full((small.nq, small.nh, small.nd), float("nan"), dtype=torch.float64, device="cuda")
    out_big = torch.full((big.nq, big.nh, big.nd), float("nan"), dtype=torch.float64, device="cuda")
    out_again = torch.full_like(out_small, float("nan"))

    # two calls in a row (the first one does the per-device set-up when this file runs alone), a larger call, then the
    # small one once more: it must not see what the larger call left in the shared array
    first = fe.omega_grid_static(small.params, small.N, small.T[0], small.q, small.h, small.delta, out_small)
    torch.cuda.synchronize()
    first = first.cpu().numpy().copy()
    second = fe.omega_grid_static(small.params, small.N, small.T[0], small.q, small.h, small.delta, out_small)
    torch.cuda.synchronize()
    second = second.cpu().numpy().copy()
    fe.omega_grid_static(big.params, big.N, big.T[0], big.q, big.h, big.delta, out_big)
    fe.omega_grid_static(small.params, small.N, small.T[0], small.q, small.h, small.delta, out_again)   # same stream: ordered
    torch.cuda.synchronize()
    third, got_big = out_again.cpu().numpy(), out_big.cpu().numpy()

    for w, got in ((small, first), (small, second), (small, third), (big, got_big)):
        assert np.all(np.isfinite(got))
        ref_default = handle_path(fe, w, w.T[0])                        # the kernel a user gets from fe_omega_grid
        ref_direct = handle_path(fe, w, w.T[0], mode=fe.EVAL_DIRECT)    # the same formulation through a handle
        assert max_rel(got, ref_default) < RTOL, (w.name, max_rel(got, ref_default))
        assert max_rel(got, ref_direct) < RTOL, (w.name, max_rel(got, ref_direct))
    # deterministic, and independent of what the array held before
    assert np.array_equal(first, second) and np.array_equal(first, third)


def test_static_entry_point_one_band_and_the_documented_example_size(fe):
    """The one-band model, and the example include/fe.h gives as fitting (N = 1024, 1 q, 16 h, 512 Delta) on a thinner
    Delta list so that the test stays short; the full example is only checked to be accepted by the limit arithmetic."""
    import torch
    w1 = W.config(1)
    out = torch.empty((w1.nq, w1.nh, w1.nd), dtype=torch.float64, device="cuda")
    fe.omega_grid_static(w1.params, w1.N, w1.T[0], w1.q, w1.h, w1.delta, out)
    torch.cuda.synchronize()
    assert max_rel(out.cpu().numpy(), handle_path(fe, w1, w1.T[0])) < RTOL
    lim = fe.static_limits()
    N, nq, nh, nd = 1024, 1, 16, 512
    assert 2 * nq + nh + nd <= lim["list"] and nq * N <= lim["trig"] and nq * nh * nd <= lim["out"]
    assert -(-N // 256) * nq * nh * nd <= lim["partial"] and lim["bytes"] <= 8 << 20
    w = W.interior_minimum(N=N, U=5.0, T=0.002, nq=nq, nh=nh, nd=32)
    out = torch.empty((w.nq, w.nh, w.nd), dtype=torch.float64, device="cuda")
    fe.omega_grid_static(w.params, w.N, w.T[0], w.q, w.h, w.delta, out)
    torch.cuda.synchronize()
    assert max_rel(out.cpu().numpy(), handle_path(fe, w, w.T[0])) < RTOL


def test_static_entry_point_leaves_free_device_memory_unchanged(fe):
    """What "allocates nothing" means for the caller, observed from outside: after the first call on the device (set-up,
    and the driver loading the kernels), the free device memory reported by the driver (cudaMemGetInfo, i.e. including
    everything outside PyTorch's pool) is the same before and after further calls -- also calls that use more of the fixed
    array than any earlier one.  The handle path, for contrast, takes memory for its scratch."""
    import torch
    small = W.ragged(seed=3, N=33, nq=2, nh=3, nd=17)
    big = W.interior_minimum(N=512, U=5.0, T=0.004, nq=2, nh=32, nd=256)     # 2 column groups x 16384 outputs of partial sums
    out_small = torch.empty((small.nq, small.nh, small.nd), dtype=torch.float64, device="cuda")
    out_big = torch.empty((big.nq, big.nh, big.nd), dtype=torch.float64, device="cuda")       # outputs are the caller's: made first
    fe.omega_grid_static(small.params, small.N, small.T[0], small.q, small.h, small.delta, out_small)    # set-up happens here at the latest
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        fe.omega_grid_static(big.params, big.N, big.T[0], big.q, big.h, big.delta, out_big)
        fe.omega_grid_static(small.params, small.N, small.T[0], small.q, small.h, small.delta, out_small)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "fe_omega_grid_static changed the device's free memory"
    assert max_rel(out_big.cpu().numpy(), handle_path(fe, big, big.T[0])) < RTOL
    with fe.FreeEnergy(big.params, big.N, big.T[0]) as F:                       # contrast: the handle path allocates scratch
        F.omega_grid(big.q, big.h, big.delta, out=out_big)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] < free0


def test_static_entry_point_refuses_what_does_not_fit(fe):
    import torch
    L = fe.lib()
    lim = fe.static_limits()
    out = torch.zeros(8, dtype=torch.float64, device="cuda")            # never written: the calls below must all be refused
    p2 = fe.make_params(W.model_params())
    p3 = fe.make_params(W.model_params(model=W.MODEL_THREE_BAND, mu=W.THREE_BAND_MU))

    def call(p, N, nq, nh, nd):
        q, h, d = np.zeros(2 * nq), np.linspace(0.0, 0.1, nh), np.linspace(0.0, 0.2, nd)
        dp = C.POINTER(C.c_double)
        rc = L.fe_omega_grid_static(C.byref(p), N, 0.01, q.ctypes.data_as(dp), nq, h.ctypes.data_as(dp), nh,
                                    d.ctypes.data_as(dp), nd, C.c_void_p(out.data_ptr()), None)
        return rc, L.fe_strerror(rc).decode()

    rc, msg = call(p2, 64, 1, 8, lim["list"])                            # list too long
    assert rc == fe.FE_EINVAL and "2 nq + nh + nd" in msg and str(lim["list"]) in msg
    rc, msg = call(p2, lim["trig"] // 2 + 1, 2, 1, 4)                    # trig tables too long
    assert rc == fe.FE_EINVAL and "nq N" in msg and str(lim["trig"]) in msg
    rc, msg = call(p2, 64, 1, 64, lim["out"] // 64 + 1)                  # too many outputs
    assert rc == fe.FE_EINVAL and "nq nh nd" in msg and str(lim["out"]) in msg
    rc, msg = call(p2, 8192, 1, 64, 512)                                 # 32 column groups x 32768 outputs of partial sums
    assert rc == fe.FE_EINVAL and "partial sums" in msg and str(lim["partial"]) in msg
    rc, msg = call(p3, 64, 1, 4, 8)                                      # three-band model
    assert rc == fe.FE_EINVAL and "three-band" in msg
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0
