"""GPU parity of the single-precision variant ("single precision implementations sometimes
offer results as good as those obtained with double precision").  precision = 32 through the same C ABI: the context
stores (rho' = q1 - 1, q2, q3) in fp32 and computes the whole step in fp32 (include/fvnl.h).  Bar (BASELINE.json
north_star): per field max|Q_gpu - Q_orc| / max|Q_orc - Q_eq| <= 1e-4 against the FP64 oracle, same metric as the fp64
tests.  All of these need a B200: -m gpu.
"""
import numpy as np
import pytest
import torch

import workloads as W
from conftest import oracle_run_cached
from helpers import oracle_from_workload, solver_from_workload, parity_error, parity_error_global

pytestmark = pytest.mark.gpu

TOL32 = 1e-4


def run32(w, steps=None, cache_key=None, rows_per_block=None):
    import paper_1311_3004_b200 as P
    steps = w.steps if steps is None else steps
    state = [a.numpy().copy() for a in w.init()]
    if cache_key is None:
        o = oracle_from_workload(w, threads=0, state=state)
        fo = o.step(steps, w.value, w.mode)
        oq, oi = o.get_state(), o.info()
    else:
        oq, oi, fo = oracle_run_cached(cache_key, w, steps)
    s = solver_from_workload(w, state=[torch.from_numpy(a) for a in state], precision=32)   # fp64 q in: the library converts
    if rows_per_block is not None:
        s.set_option(P.OPT_ROWS_PER_BLOCK, rows_per_block)
    fg = s.step(steps, w.value, w.mode)
    gq = [a.cpu().numpy() for a in s.get_state(as_q64=True)]
    return gq, oq, s.info(), oi, fg, fo


def check32(w, steps=None, tol=TOL32, metric=parity_error, **kw):
    gq, oq, gi, oi, fg, fo = run32(w, steps, **kw)
    assert fg == fo == 0, (fg, fo)
    assert gi["steps"] == oi["steps"]
    for k in ("t", "dt", "M", "cfl"):
        assert gi[k] == pytest.approx(oi[k], rel=2e-6), k            # the speeds that enter M are fp32
    err = metric(gq, oq)
    print(f"PARITY32 {w.name} {w.nx}x{w.ny} steps={gi['steps']} err={err:.3e} tol={tol:g}")
    assert err <= tol, f"{w.name}: fp32 parity error {err:.3e} > {tol}"
    return err


def test_fp32_c1_piston_full():
    """C1 at full size (512 x 4, 2000 steps): plane piston, q3 == 0 exactly also in fp32."""
    check32(W.c1_piston())


def test_fp32_c2_small_and_full():
    check32(W.c2_pulse(n=300, ny=200, sigma_cells=8.0, steps=150))
    check32(W.c2_pulse(), cache_key="C2")


def test_fp32_c3_small_and_full():
    check32(W.c3_random(n=517, ny=263, steps=200, sig_lo=3.0, sig_hi=20.0))
    check32(W.c3_random(), cache_key="C3")


def test_fp32_c4_small_packet_and_cw():
    check32(W.c4_hifu(nx=640, ny=256, steps=400, focus_cells=160.0, aperture_cells=80.0, tau0=-4.5))
    check32(W.c4_hifu(nx=320, ny=192, steps=300, focus_cells=120.0, aperture_cells=60.0, tau0=0.0, shape=W.SINE))


def test_fp32_c5_small_and_2048():
    check32(W.c5_sweep(n=256, steps=100))
    check32(W.c5_sweep(n=1000, ny=96, steps=100))
    check32(W.c5_sweep(n=2048), cache_key="C5-2048")


@pytest.mark.parametrize("rows", [4, 7, 64])
def test_fp32_forced_chunk_heights(rows):
    check32(W.c3_random(n=300, ny=131, steps=25, sig_lo=3.0, sig_hi=12.0), rows_per_block=rows)
    check32(W.c4_hifu(nx=260, ny=90, steps=40, focus_cells=60.0, aperture_cells=30.0, tau0=-1.0), rows_per_block=rows)


def test_fp32_edges_and_tiny_grids():
    """REFLECT / EXTRAP / PERIODIC, dx != dy, fixed dt on the minimum grid, sources on other sides."""
    import paper_1311_3004_b200 as P
    w = W.c2_pulse(n=200, ny=150, sigma_cells=6.0, steps=200)
    w.bc = [(P.REFLECT, None), (P.EXTRAP, None), (P.EXTRAP, None), (P.REFLECT, None)]
    w.dy = w.dx * 1.25
    check32(w)
    for nx, ny in ((4, 4), (5, 4), (33, 5)):
        for bc in (P.PERIODIC, P.EXTRAP, P.REFLECT):
            w = W.c3_random(n=nx, ny=ny, steps=20, sig_lo=1.0, sig_hi=2.0, seed=7 + nx * ny)
            w.bc = [(bc, None)] * 4
            w.mode, w.value = 0, 0.4 * w.dx / w.medium["c0"]
            check32(w)
    dx = W.LAMBDA_1MHZ / 32
    base = dict(shape=P.PACKET, amp=4e-4, freq_hz=1e6, focus_m=50 * dx, centre_m=70 * dx, half_aperture_m=30 * dx,
                t0_s=-1.5e-6, steep=0.0)
    w = W.c2_pulse(n=150, ny=170, sigma_cells=5.0, steps=120, amp=2e-4)
    w.bc = [(P.EXTRAP, None), (P.SOURCE, dict(base)), (P.SOURCE, dict(base, shape=P.SINE, focus_m=0.0, half_aperture_m=0.0, t0_s=0.0)),
            (P.SOURCE, dict(base, shape=P.SINE, t0_s=0.0, centre_m=80 * dx))]
    check32(w)


def test_fp32_taylor_1e7_perturbation():
    """C1-T: a 1e-7 perturbation on a unit background -- one ulp of 1.0f is 1.2e-7, so an fp32 code that stores q1 cannot
    even represent this wave.  In perturbation form it is resolved like any other: the same 1e-4 bar (one scale for all
    fields: q3 is round-off here, as in the fp64 test)."""
    w = W.c1t_taylor(eta=10, nu_w=0.9, y_periodic=True)
    check32(w, steps=400, metric=parity_error_global)


def test_fp32_own_form_io_restart_and_flags():
    """float32 planes (rho', q2, q3) in and out (host and device), bitwise restart, the sticky flags, equilibrium."""
    import paper_1311_3004_b200 as P
    w = W.c3_random(n=200, ny=120, steps=40, sig_lo=3.0, sig_hi=10.0)
    q = w.init()
    own = [(q[0] - 1.0).float(), q[1].float(), q[2].float()]
    a = solver_from_workload(w, state=own, precision=32)                    # host float planes
    a.step(40, w.value, 1)
    ref = [x.clone() for x in a.get_state()]
    assert ref[0].dtype == torch.float32 and float(ref[0].abs().max()) < 1e-2     # rho', not q1
    b = solver_from_workload(w, state=[x.cuda() for x in own], precision=32)
    b.step(15, w.value, 1)
    mid = b.get_state(host=True)
    info = b.info()
    c = solver_from_workload(w, state=mid, precision=32)
    c.set_clock(info["t"], info["M"])
    c.step(25, w.value, 1)
    for x, y in zip(ref, c.get_state()):
        assert torch.equal(x, y)
    # flags as in fp64
    w2 = W.c2_pulse(n=64, steps=3)
    w2.value = 1.3
    s = solver_from_workload(w2, precision=32)
    assert s.step(3, 1.3, 1) & P.ECFL
    s = P.Solver(150, 37, 1e-4, 1e-4, c0=1500.0, rho0=1000.0, beta=3.5, delta=4.3e-6, precision=32)
    for side in range(4):
        s.set_bc(side, P.PERIODIC)
    assert s.step(25, 0.9, 1) == 0
    r, m2, m3 = s.get_state()
    assert not r.any() and not m2.any() and not m3.any()
    assert s.info()["M"] == pytest.approx(1e4, rel=1e-7)
    with pytest.raises(P.FvnlError):
        s.set_option(P.OPT_KERNEL, P.KERNEL_UNFUSED)                         # comparison paths are fp64 only


def test_fp32_c5_16384_windows():
    """C5 at 16384^2 in fp32 over the full 100 steps (the configuration bench.py --precision 32 times): two windows the
    FP64 oracle recomputes cell by cell, fixed dt."""
    import paper_1311_3004_b200 as P
    from test_gpu_parity import _window_oracle_rect
    n = 16384
    w = W.c5_sweep(n=n)
    q0 = w.init(device="cuda")
    s = P.Solver(w.nx, w.ny, w.dx, w.dy, **w.medium, precision=32)
    for side, (kind, src) in enumerate(w.bc):
        s.set_bc(side, kind, src)
    s.set_state(*q0)
    dt = w.value * w.dx / (w.medium["c0"] * 1.004)
    assert s.step(100, dt, 0) == 0
    out = s.get_state()
    worst = 0.0
    for (i0, j0, wx, wy) in ((n - 24, n - 24, 48, 48), (122 * 31 - 24, 377, 48, 720)):
        ref, (ii, jj) = _window_oracle_rect(w, q0, i0, j0, wx, wy, 308, 100, dt)
        got = [o_[torch.as_tensor(jj, device="cuda")][:, torch.as_tensor(ii, device="cuda")].double().cpu().numpy() for o_ in out]
        got[0] = got[0] + 1.0
        err = parity_error(got, ref)
        print(f"PARITY32 C5-{n} window ({i0},{j0}) {wx}x{wy} steps=100 err={err:.3e} tol={TOL32:g}")
        worst = max(worst, err)
    assert worst <= TOL32


def test_fp32_oblique_taylor_and_moving_domain():
    """The two other 'next' rows in fp32: oblique Taylor shock and the moving domain."""
    import math
    w = W.c1t_taylor(eta=10, nu_w=0.9, x_lo=-4.0, x_hi=10.0, y_lo=-5.0, y_hi=8.0, theta=math.pi / 8)
    check32(w, steps=90, metric=parity_error_global)
    w = W.c2_pulse(n=260, ny=90, sigma_cells=6.0, steps=1, amp=1e-3)
    state = [a.numpy().copy() for a in w.init()]
    o = oracle_from_workload(w, threads=0, state=state)
    s = solver_from_workload(w, state=[torch.from_numpy(a) for a in state], precision=32)
    for n, k in ((7, 1), (5, 3), (11, 2), (9, 1)):
        assert o.step(n, 0.9, 1) == 0 and s.step(n, 0.9, 1) == 0
        o.shift(k)
        s.shift(k)
    assert o.step(6, 0.9, 1) == 0 and s.step(6, 0.9, 1) == 0
    err = parity_error([a.cpu().numpy() for a in s.get_state(as_q64=True)], o.get_state())
    print(f"PARITY32 moving pulse err={err:.3e}")
    assert err <= TOL32
