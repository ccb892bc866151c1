"""dg_drag_update_host_static (include/dg.h): the host-buffer update for callers that cannot allocate device memory.

Who that is: a simulation code whose own memory pool took the whole GPU at start-up (a cudaMalloc from a library
would simply fail), a time-step loop that cannot accept the device-wide stall cudaMalloc / cudaFree cause, a process
under a device-memory quota, a plug-in whose host forbids allocation after initialisation.  The entry point stages the
cells in a fixed 32 MiB array that is part of libdg.so instead of asking the runtime for memory.

What is checked here: that it returns the same bits as the existing, allocating path (dg_drag_update_host) — the
tolerance the other host-path tests use is bit equality, tests/test_gpu_parity.py — on calls made back to back, because
every call shares that one array and finds the previous call's bytes in it; and that sizes beyond the array are refused
with a clear error before anything is touched.

This file is named so that pytest collects it last (`pytest --collect-only -q`): with `-x` a failure here cannot hide a
test that would have run after it.  It does not rely on what ran before: it passes alone in a fresh process, where
its first call is the one that resolves the array's device address, and after the rest of the suite.
"""
import ctypes as C

import pytest
import torch

from paper_2509_25347_b200 import workloads as W


def max_cells(dg, N):
    return dg.DG_STATIC_STAGE_BYTES // (8 * (8 * N + 7))


def test_oversized_and_malformed_requests_are_refused_before_any_cuda_call(dg):
    """Runs without a GPU: the capacity and argument checks come before the first CUDA call."""
    lib = dg.raw()
    buf = (C.c_double * 64)()
    p = C.addressof(buf)
    f = lib.dg_drag_update_host_static
    assert max_cells(dg, 1) == 279620 and max_cells(dg, 8) == 59074 and max_cells(dg, 16) == 31068   # as documented
    for N in (1, 8, 16):
        assert f(p, p, p, 0.1, p, N, max_cells(dg, N) + 1, p, None) == dg.DG_ECAPACITY
        assert f(p, p, p, 0.1, p, N, 2 ** 40, p, None) == dg.DG_ECAPACITY
    msg = lib.dg_status_string(dg.DG_ECAPACITY).decode()
    assert msg.startswith("DG_ECAPACITY") and "dg_drag_update_host_static" in msg and "32 MiB" in msg
    assert f(p, p, p, 0.1, p, 0, 8, p, None) == dg.DG_ERANGE
    assert f(p, p, p, 0.1, p, 17, 8, p, None) == dg.DG_ERANGE
    assert f(p, p, p, 0.1, p, 4, -1, p, None) == dg.DG_ERANGE
    assert f(p, p, p, float("nan"), p, 4, 8, p, None) == dg.DG_EINVAL
    assert f(p, p, p, -1.0, p, 4, 8, p, None) == dg.DG_EINVAL
    assert f(p, p, p, 0.1, p, 4, 8, None, None) == dg.DG_ENULL
    assert f(p, p, p, 0.1, p + 4, 4, 8, p, None) == dg.DG_EALIGN
    assert f(None, None, None, 0.1, None, 4, 0, None, None) == dg.DG_OK          # ncells = 0: no-op


@pytest.mark.gpu
def test_static_staging_gives_the_bits_of_the_allocating_host_path_on_back_to_back_calls(dg, cuda):
    """Calls in a row with different N, sizes and inputs, so that each call lays its fields over different, stale bytes
    of the shared array (a 16-species problem, then a larger 4-species one, then the first again, then one that fills
    the array to the last cell it accepts); each must equal dg_drag_update_host bit for bit, also with pageable memory
    and in place."""
    cases = [(16, 1237, 11), (4, 10007, 12), (16, 1237, 11), (8, max_cells(dg, 8), 13), (1, 5000, 14)]
    want = {}
    for N, ncells, seed in cases:                     # the existing path first, on its own
        wl = W.make_workload(5, ncells=ncells, N=N, device="cpu", seed=seed)
        want[(N, ncells, seed)] = (wl, dg.dg_drag_update_host(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in))
    dg.dg_host_release()
    for N, ncells, seed in cases:                     # then the new entry point, call after call
        wl, ref = want[(N, ncells, seed)]
        assert torch.isfinite(ref).all() and not torch.equal(ref, wl.p_in)
        out = dg.dg_drag_update_host_static(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in)
        assert torch.equal(out, ref), (N, ncells)
        # the same call again straight away: its own previous contents are what it now finds in the array
        pinned = [t.pin_memory() for t in (wl.rho_g, wl.rho_d, wl.t_s, wl.p_in)]
        out2 = dg.dg_drag_update_host_static(pinned[0], pinned[1], pinned[2], wl.dt, pinned[3])
        assert torch.equal(out2, ref), (N, ncells)
        p = wl.p_in.clone()                           # in place: p_out aliases p_in
        dg.dg_drag_update_host_static(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, p, p_out=p)
        assert torch.equal(p, ref), (N, ncells)
    # and it agrees with the device entry point on device buffers
    wl, ref = want[cases[1]]
    dev = dg.dg_drag_update(wl.rho_g.to(cuda), wl.rho_d.to(cuda), wl.t_s.to(cuda), wl.dt, wl.p_in.to(cuda))
    assert torch.equal(dev.cpu(), ref)


@pytest.mark.gpu
def test_a_refused_call_leaves_the_output_alone_and_the_next_call_works(dg, cuda):
    N = 16
    ncells = max_cells(dg, N) + 1
    wl = W.make_workload(5, ncells=ncells, N=N, device="cpu", seed=21)
    out = torch.full_like(wl.p_in, -7.0)
    with pytest.raises(dg.DgError) as err:
        dg.dg_drag_update_host_static(wl.rho_g, wl.rho_d, wl.t_s, wl.dt, wl.p_in, p_out=out)
    assert err.value.status == dg.DG_ECAPACITY and "DG_ECAPACITY" in str(err.value)
    assert (out == -7.0).all()
    # one cell fewer fits, on a non-default stream too
    k = ncells - 1
    sub = [wl.rho_g[:k].contiguous(), wl.rho_d[:, :k].contiguous(), wl.t_s[:, :k].contiguous(),
           wl.p_in[:, :, :k].contiguous()]
    ref = dg.dg_drag_update_host(sub[0], sub[1], sub[2], wl.dt, sub[3])
    with torch.cuda.stream(torch.cuda.Stream()):
        got = dg.dg_drag_update_host_static(sub[0], sub[1], sub[2], wl.dt, sub[3])
    assert torch.equal(got, ref)
    dg.dg_host_release()
