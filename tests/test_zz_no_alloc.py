"""fvnl_step_noalloc: the allocation-free entry point (include/fvnl.h) against the existing path.

One fixed-dt step of the three-pass kernels whose scratch (clock block, Q*, Q**) lives in a 16 MiB file-scope device array
instead of cudaMalloc'ed memory, for callers that cannot allocate (CUDA graph capture, serving loops).  Checked here against
the context-based path (fvnl_create / fvnl_step, default kernel) on the same seeded inputs, on TWO CALLS IN A ROW -- the
array is shared by every call and keeps the previous call's contents -- with the parity metric and the 1e-10 bar of
tests/test_gpu_parity.py; against the three-pass kernels of the context path, which run the same arithmetic, the result must
be bitwise identical.  This file sorts last on purpose (the suite runs with pytest -x).
"""
import numpy as np
import pytest
import torch

import workloads as W
from helpers import solver_from_workload, parity_error

pytestmark = pytest.mark.gpu

TOL = 1e-10


def noalloc_steps(P, w, state, dt, nsteps, t0=0.0):
    """nsteps calls of fvnl_step_noalloc in a row, ping-ponging between two caller-owned states.  Returns (state, flag words)."""
    med = P.fvnl_medium(w.medium["c0"], w.medium["rho0"], w.medium["beta"], w.medium["delta"])
    kinds = [k for k, _ in w.bc]
    srcs = [None if s is None else (s if isinstance(s, P.fvnl_source) else P.fvnl_source(**s)) for _, s in w.bc]
    a = [x.clone() for x in state]
    b = [torch.empty_like(x) for x in state]
    flags = torch.full((nsteps,), -1, dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    t = t0
    for n in range(nsteps):
        rc = P.fvnl_step_noalloc(w.nx, w.ny, w.dx, w.dy, med, kinds, srcs, t, dt, [x.data_ptr() for x in a],
                                 [x.data_ptr() for x in b], flags[n:].data_ptr(), stream)
        assert rc == P.OK, P.fvnl_strerror(rc)
        a, b = b, a
        t = t + dt                                     # (the context path adds dt to t the same way)
    torch.cuda.synchronize()
    return a, flags.cpu().tolist()


def context_steps(P, w, state, dt, nsteps, unfused):
    s = solver_from_workload(w, state=[x.clone() for x in state])
    if unfused:
        s.set_option(P.OPT_KERNEL, P.KERNEL_UNFUSED)
    assert s.step(nsteps, dt, 0) == 0
    out = [x.clone() for x in s.get_state()]
    s.close()
    return out


def cases(P):
    dx = W.c3_random(n=64, ny=64).dx
    w1 = W.c3_random(n=300, ny=217, steps=2, sig_lo=3.0, sig_hi=12.0)                   # periodic
    w2 = W.c2_pulse(n=180, ny=140, sigma_cells=5.0, steps=2, amp=2e-4)                  # focused source, reflect, extrapolation
    w2.bc = [(P.SOURCE, dict(shape=P.SINE, amp=2e-4, freq_hz=1.0e6, focus_m=40 * dx, centre_m=70 * dx,
                              half_aperture_m=30 * dx, t0_s=0.0, steep=0.0)),
             (P.EXTRAP, None), (P.REFLECT, None), (P.EXTRAP, None)]
    return [w1, w2]


def test_noalloc_matches_the_context_path_on_two_calls_in_a_row():
    import paper_1311_3004_b200 as P
    for w in cases(P):
        dt = 0.8 * w.dx / (w.medium["c0"] * 1.01)
        state = [x.to("cuda") for x in w.init()]
        ref1 = context_steps(P, w, state, dt, 1, unfused=False)
        ref2 = context_steps(P, w, state, dt, 2, unfused=False)
        same2 = context_steps(P, w, state, dt, 2, unfused=True)
        out1, f1 = noalloc_steps(P, w, state, dt, 1)
        out2, f2 = noalloc_steps(P, w, state, dt, 2)             # calls no. 2 and 3 on the shared array
        assert f1 == [0] and f2 == [0, 0]
        e1 = parity_error([x.cpu().numpy() for x in out1], [x.cpu().numpy() for x in ref1])
        e2 = parity_error([x.cpu().numpy() for x in out2], [x.cpu().numpy() for x in ref2])
        print(f"PARITY noalloc {w.name} {w.nx}x{w.ny} after 1 / 2 calls: {e1:.3e} / {e2:.3e} tol={TOL:g}")
        assert e1 <= TOL and e2 <= TOL
        for g, r in zip(out2, same2):                             # same kernels, same arithmetic: bit for bit
            assert torch.equal(g, r)
    # a smaller grid right after a larger one: stale contents of the array beyond the new layout must not matter
    w = W.c3_random(n=64, ny=40, steps=1, sig_lo=2.0, sig_hi=6.0)
    dt = 0.8 * w.dx / (w.medium["c0"] * 1.01)
    state = [x.to("cuda") for x in w.init()]
    out, f = noalloc_steps(P, w, state, dt, 2)
    ref = context_steps(P, w, state, dt, 2, unfused=True)
    assert f == [0, 0] and all(torch.equal(g, r) for g, r in zip(out, ref))


def test_noalloc_flags_and_limits():
    import paper_1311_3004_b200 as P
    w = W.c3_random(n=64, ny=40, steps=1, sig_lo=2.0, sig_hi=6.0)
    state = [x.to("cuda") for x in w.init()]
    # a step that runs with nu > 1 reports FVNL_ECFL through the device flag word, and the next call starts clean again
    _, f = noalloc_steps(P, w, state, 1.3 * w.dx / w.medium["c0"], 1)
    assert f[0] & 16
    _, f = noalloc_steps(P, w, state, 0.5 * w.dx / w.medium["c0"], 1)
    assert f == [0]
    med = P.fvnl_medium(1500.0, 1000.0, 3.5, 4.3e-6)
    tq, to = (torch.ones(3, 8, device="cuda", dtype=torch.float64) for _ in range(2))      # (kept alive: distinct addresses)
    q, o = [x.data_ptr() for x in tq], [x.data_ptr() for x in to]
    kinds = [P.PERIODIC] * 4
    # beyond the static array: rejected before anything is launched (the 8-element buffers are never touched)
    assert 6 * 600 * 600 * 8 > P.NOALLOC_MAX_BYTES
    assert P.fvnl_step_noalloc(600, 600, 1e-4, 1e-4, med, kinds, None, 0.0, 1e-8, q, o) == P.ESIZE
    assert "fvnl_step_noalloc" in P.fvnl_strerror(P.ESIZE)
    assert P.fvnl_step_noalloc(580, 580, 1e-4, 1e-4, med, [P.PERIODIC, P.EXTRAP, P.EXTRAP, P.EXTRAP], None, 0.0, 1e-8, q, o) == P.EARG
    assert P.fvnl_step_noalloc(64, 40, 1e-4, 1e-4, med, kinds, None, 0.0, 1e-8, q, q) == P.EARG          # in == out
    assert P.fvnl_step_noalloc(64, 40, 1e-4, 1e-4, med, [P.SOURCE, P.EXTRAP, P.EXTRAP, P.EXTRAP], None, 0.0, 1e-8, q, o) == P.EARG
