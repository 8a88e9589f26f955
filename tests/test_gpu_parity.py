"""GPU parity: the CUDA path (through the C ABI, paper_1311_3004_b200) against the CPU oracle, element by element,
on the same seeded inputs.  Bar (BASELINE.json north_star / SURVEY.md 8(d)): per field
E^m = max|Q_gpu - Q_orc| / max|Q_orc - Q_eq| <= 1e-10 after the full step count of the case; a field that is
identically at equilibrium in the oracle must be so on the GPU.  All of these need a B200: -m gpu.
"""
import numpy as np
import pytest
import torch

import workloads as W
from conftest import read_golden_kv
from helpers import oracle_from_workload, solver_from_workload, parity_error, parity_error_global

pytestmark = pytest.mark.gpu

TOL = 1e-10


def run_both(w, steps=None, kernel=None, rows_per_block=None, chunks=None, cache_key=None):
    """Advance oracle and GPU over `steps` (split in `chunks` fvnl_step calls on the GPU side); returns states + infos.
    cache_key: share the oracle's run of a full-size workload with the other tests of the session."""
    import paper_1311_3004_b200 as P
    from conftest import oracle_run_cached
    steps = w.steps if steps is None else steps
    state = [a.numpy().copy() for a in w.init()]
    if cache_key is not None:
        oq, oi, fo = oracle_run_cached(cache_key, w, steps)
        s = solver_from_workload(w, state=[torch.from_numpy(a) for a in state])
        fg = s.step(steps, w.value, w.mode)
        return [a.cpu().numpy() for a in s.get_state()], oq, s.info(), oi, fg, fo
    o = oracle_from_workload(w, threads=0, state=state)
    fo = o.step(steps, w.value, w.mode)
    s = solver_from_workload(w, state=[torch.from_numpy(a) for a in state])
    if kernel is not None:
        select(s, kernel)
    if rows_per_block is not None:
        s.set_option(P.OPT_ROWS_PER_BLOCK, rows_per_block)
    fg = 0
    for part in (chunks or [steps]):
        fg |= s.step(part, w.value, w.mode)
    gq = [a.cpu().numpy() for a in s.get_state()]
    return gq, o.get_state(), s.info(), o.info(), fg, fo


def select(s, kernel):
    """kernel = (FVNL_OPT_KERNEL value, FVNL_OPT_VARIANT value, FVNL_OPT_SMALL_GRID value)."""
    import paper_1311_3004_b200 as P
    s.set_option(P.OPT_KERNEL, kernel[0])
    s.set_option(P.OPT_VARIANT, kernel[1])
    s.set_option(P.OPT_SMALL_GRID, kernel[2])


def check(w, steps=None, tol=TOL, metric=parity_error, **kw):
    gq, oq, gi, oi, fg, fo = run_both(w, steps, **kw)
    assert fg == fo == 0, (fg, fo)
    assert gi["steps"] == oi["steps"]
    assert gi["t"] == pytest.approx(oi["t"], rel=1e-12)
    assert gi["dt"] == pytest.approx(oi["dt"], rel=1e-12)
    assert gi["M"] == pytest.approx(oi["M"], rel=1e-12)
    assert gi["cfl"] == pytest.approx(oi["cfl"], rel=1e-12)
    err = metric(gq, oq)
    print(f"PARITY {w.name} {w.nx}x{w.ny} steps={gi['steps']} kernel={kw.get('kernel')} err={err:.3e} tol={tol:g}")
    assert err <= tol, f"{w.name}: parity error {err:.3e} > {tol}"
    return err


# (FVNL_OPT_KERNEL, FVNL_OPT_VARIANT, FVNL_OPT_SMALL_GRID): the warp-specialised one-pass kernel k_step_ws (for every kind of
# edge; analytic SOURCE cells come from the boundary kernel / the step kernel's tail), the single-role one-pass kernel
# k_step_fused (evaluates them in place), and the three-pass comparison kernels -- each with one launch per step -- and
# "cluster": the library's default behaviour, in which a grid of at most 16384 cells runs all steps of a call in one launch
# of one thread-block cluster (k_steps_cluster, fvnl_small.cuh; larger grids take the "ws" path there too)
KERNELS = [(0, 0, 0), (0, 1, 0), (1, 0, 0), (0, 0, 1)]
KIDS = ["ws", "fused", "unfused", "cluster"]


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_p9_4x4_worked_step(kernel):
    """The 4x4 worked step of SURVEY.md 8(c) (tests/golden/p9_4x4.txt, written from an independent prototype of the
    same reading and reproduced by the oracle): periodic and extrapolation edges, fixed dt, source step on."""
    import paper_1311_3004_b200 as P
    g = read_golden_kv("p9_4x4.txt")
    i, j = np.meshgrid(np.arange(4), np.arange(4))
    q1 = 1 + 0.01 * (((3 * i + 5 * j * j + i * j) % 7) - 3) / 3
    q2 = 0.002 * (((2 * i + 3 * j) % 5) - 2)
    q3 = 0.003 * (((i * i + j) % 4) - 1.5)
    for bc, keys in ((P.PERIODIC, True), (P.EXTRAP, False)):
        s = P.Solver(4, 4, 1.0, 1.0, c0=1.0, rho0=1.0, beta=3.5, delta=0.05)
        select(s, kernel)
        for side in range(4):
            s.set_bc(side, bc)
        s.set_state(torch.from_numpy(q1), torch.from_numpy(q2.astype(float)), torch.from_numpy(q3))
        assert s.step(1, 0.5, 0) == 0
        out = [a.cpu().numpy() for a in s.get_state()]
        if keys:
            for m, name in enumerate(("q1", "q2", "q3")):
                assert np.abs(out[m] - np.array(g[name])).max() <= 1e-13
            assert s.info()["M"] == pytest.approx(g["M"][0][0], rel=1e-13)
        else:
            c00 = np.array([out[m][0, 0] for m in range(3)])
            c33 = np.array([out[m][3, 3] for m in range(3)])
            assert np.abs(c00 - np.array(g["extrap_cell_0_0"][0])).max() <= 1e-13
            assert np.abs(c33 - np.array(g["extrap_cell_3_3"][0])).max() <= 1e-13


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_c1_piston_full(kernel):
    """C1 at full size: 512x4, 2000 steps, plane piston on x-lo, extrapolation x-hi, periodic y; q3 == 0 exactly."""
    check(W.c1_piston(), kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_c2_pulse_small(kernel):
    """C2 scaled to 300 x 200 (ragged against every tile size), sigma 8 cells, extrapolation edges, 150 steps:
    the pulse reaches and leaves through the edges."""
    check(W.c2_pulse(n=300, ny=200, sigma_cells=8.0, steps=150), kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_c3_random_small(kernel):
    """C3 scaled to 517 x 263 (prime-ish, several strips with a ragged tail), periodic, 200 steps as the full config."""
    check(W.c3_random(n=517, ny=263, steps=200, sig_lo=3.0, sig_hi=20.0), kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_c4_hifu_small(kernel):
    """C4 scaled: 640 x 256, focus at 160 cells, aperture 80 cells, 400 steps (packet enters, focuses, nonlinear)."""
    w = W.c4_hifu(nx=640, ny=256, steps=400, focus_cells=160.0, aperture_cells=80.0, tau0=-4.5)
    check(w, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_c4_cw_source_small(kernel):
    """The continuous-wave reading of "time-harmonic" (SINE with an aperture and a focus)."""
    w = W.c4_hifu(nx=320, ny=192, steps=300, focus_cells=120.0, aperture_cells=60.0, tau0=0.0, shape=W.SINE)
    check(w, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_c5_small_sizes(kernel):
    """C5 generator at 256^2 and 1000 x 96, nu_W = 0.9, 100 steps."""
    check(W.c5_sweep(n=256, steps=100), kernel=kernel)
    check(W.c5_sweep(n=1000, ny=96, steps=100), kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_taylor_dirichlet_edges(kernel):
    """C1-T (eta = 10): analytic (41) cells on all four sides, and with periodic y-edges.  The perturbation is 1e-7
    of the unit background, so one ulp of the state is already 2e-9 of it: the bar is 1e-7 (SURVEY.md 8(d) C1-T
    note), on one scale for all fields -- q3 is ~1e-11 here (round-off and edge mismatch), see parity_error_global."""
    for yper in (False, True):
        w = W.c1t_taylor(eta=10, nu_w=0.9, y_periodic=yper)
        check(w, steps=400, tol=1e-7, metric=parity_error_global, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_reflecting_and_mixed_edges(kernel):
    """REFLECT on x-lo and y-hi, EXTRAP elsewhere, off-centre pulse, non-square cells (dx != dy)."""
    import paper_1311_3004_b200 as P
    w = W.c2_pulse(n=200, ny=150, sigma_cells=6.0, steps=200)
    w.bc = [(P.REFLECT, None), (P.EXTRAP, None), (P.EXTRAP, None), (P.REFLECT, None)]
    w.dy = w.dx * 1.25
    base = w.init

    def init(device="cpu"):
        q1, q2, q3 = base(device)
        return torch.roll(q1, shifts=(40, -60), dims=(0, 1)), q2, q3
    w.init = init
    check(w, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_fixed_dt_mode_and_tiny_grids(kernel):
    """mode 0 (fixed dt) on the minimum grid 4x4 and on 5 x 4 / 4 x 7, periodic and extrapolation."""
    import paper_1311_3004_b200 as P
    for nx, ny in ((4, 4), (5, 4), (4, 7), (33, 5)):
        for bc in (P.PERIODIC, P.EXTRAP, P.REFLECT):
            w = W.c3_random(n=nx, ny=ny, steps=20, sig_lo=1.0, sig_hi=2.0, seed=7 + nx * ny)
            w.bc = [(bc, None)] * 4
            w.mode, w.value = 0, 0.4 * w.dx / w.medium["c0"]
            check(w, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_restart_is_bitwise(kernel):
    """P10: N steps == k steps + get_state/get_info + set_state/set_clock + (N-k) steps, bit for bit; and splitting
    one fvnl_step call into several changes nothing."""
    import paper_1311_3004_b200 as P
    w = W.c3_random(n=200, ny=120, steps=40, sig_lo=3.0, sig_hi=10.0)
    a = solver_from_workload(w)
    select(a, kernel)
    a.step(40, w.value, 1)
    ref = [x.clone() for x in a.get_state()]
    b = solver_from_workload(w)
    select(b, kernel)
    b.step(10, w.value, 1)
    b.step(5, w.value, 1)
    mid = [x.clone() for x in b.get_state(host=True)]
    info = b.info()
    c = solver_from_workload(w)
    select(c, kernel)
    c.set_state(*mid)
    c.set_clock(info["t"], info["M"])
    c.step(25, w.value, 1)
    for x, y in zip(ref, c.get_state()):
        assert torch.equal(x, y)
    assert c.info()["t"] == a.info()["t"]


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_mixed_modes_and_unknown_M_restart(kernel):
    """Which M the first CFL-mode step uses (include/fvnl.h, reading A7; the oracle's rule is `M_prev > 0`): after
    set_state -> step(mode 0) it is the M of that fixed-dt step, NOT a pre-pass; after set_clock(t, 0) it is the pre-pass
    on the current state alone (no maximum left over from earlier steps)."""
    w = W.c2_pulse(n=96, ny=80, sigma_cells=5.0, steps=1, amp=5e-3)
    state = [a.numpy().copy() for a in w.init()]
    dt0 = 0.3 * w.dx / w.medium["c0"]
    # (a) fixed dt, then CFL mode
    o = oracle_from_workload(w, threads=0, state=state)
    s = solver_from_workload(w, state=[torch.from_numpy(a) for a in state])
    select(s, kernel)
    assert o.step(7, dt0, 0) == 0 and s.step(7, dt0, 0) == 0
    assert o.step(9, 0.9, 1) == 0 and s.step(9, 0.9, 1) == 0
    for k in ("t", "dt", "M", "cfl"):
        assert s.info()[k] == pytest.approx(o.info()[k], rel=1e-12), k
    assert parity_error([a.cpu().numpy() for a in s.get_state()], o.get_state()) <= TOL
    # (b) the pulse has spread: M now is smaller than at the start.  Forget M on both sides -> pre-pass on the current state
    t = o.info()["t"]
    o.set_clock(t, 0.0)
    s.set_clock(t, 0.0)
    assert o.step(1, 0.9, 1) == 0 and s.step(1, 0.9, 1) == 0
    assert s.info()["dt"] == pytest.approx(o.info()["dt"], rel=1e-12)
    assert o.step(5, 0.9, 1) == 0 and s.step(5, 0.9, 1) == 0
    assert parity_error([a.cpu().numpy() for a in s.get_state()], o.get_state()) <= TOL
    # (c) a state with a much larger M first, then set_state of a quiet one: nothing of the old maximum survives
    loud = [state[0] + 0.05 * (state[0] - 1.0) / 5e-3, state[1], state[2]]
    o2 = oracle_from_workload(w, threads=0, state=loud)
    s2 = solver_from_workload(w, state=[torch.from_numpy(a) for a in loud])
    select(s2, kernel)
    assert o2.step(2, 0.9, 1) == 0 and s2.step(2, 0.9, 1) == 0
    o2.set_state(*state)
    s2.set_state(*[torch.from_numpy(a) for a in state])
    assert o2.step(3, 0.9, 1) == 0 and s2.step(3, 0.9, 1) == 0
    assert s2.info()["dt"] == pytest.approx(o2.info()["dt"], rel=1e-12)
    assert parity_error([a.cpu().numpy() for a in s2.get_state()], o2.get_state()) <= TOL


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_run_to_run_determinism(kernel):
    import paper_1311_3004_b200 as P
    w = W.c3_random(n=300, ny=300, steps=30, sig_lo=3.0, sig_hi=10.0)
    outs = []
    for _ in range(2):
        s = solver_from_workload(w)
        select(s, kernel)
        s.step(30, w.value, 1)
        outs.append([x.clone() for x in s.get_state()])
    for x, y in zip(*outs):
        assert torch.equal(x, y)


def test_fused_equals_unfused_to_rounding():
    """Two independently structured GPU implementations of the same arithmetic agree to a few ulp of the state."""
    import paper_1311_3004_b200 as P
    w = W.c3_random(n=700, ny=300, steps=50, sig_lo=3.0, sig_hi=20.0)
    outs = []
    for kernel in KERNELS:
        s = solver_from_workload(w)
        select(s, kernel)
        assert s.step(50, w.value, 1) == 0
        outs.append([x.cpu().numpy() for x in s.get_state()])
    assert parity_error(outs[0], outs[2]) <= 1e-11
    assert parity_error(outs[1], outs[2]) <= 1e-11


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_flags(kernel):
    """nu_W > 1 sets FVNL_ECFL; a state outside the real-eigenvalue region S sets FVNL_ENONREAL
    (PAPER.md:263-267); q1 <= 0 sets FVNL_ENONPOS -- same words as the oracle."""
    import paper_1311_3004_b200 as P
    w = W.c2_pulse(n=64, steps=3)
    w.value = 1.3
    gq, oq, gi, oi, fg, fo = run_both(w, kernel=kernel)
    assert fg & P.ECFL and fo & P.ECFL
    w = W.c2_pulse(n=64, steps=1)
    base = w.init

    def init(device="cpu"):
        q1, q2, q3 = base(device)
        q2 = q2.clone()
        q2[10:20, 10:20] = 1.5          # (u/c0)^2 far above S(rho/rho0 ~ 1) = 1
        return q1, q2, q3
    w.init = init
    w.mode, w.value = 0, 1e-10
    gq, oq, gi, oi, fg, fo = run_both(w, kernel=kernel)
    assert fo & P.ENONREAL and fg & P.ENONREAL


def test_api_errors():
    import paper_1311_3004_b200 as P
    med = P.fvnl_medium(1500.0, 1000.0, 3.5, 4.3e-6)
    rc, h = P.fvnl_create(3, 8, 1e-4, 1e-4, med)
    assert rc == P.EARG
    rc, h = P.fvnl_create(8, 8, 1e-4, 1e-4, med, precision=16)
    assert rc == P.EARG
    rc, h = P.fvnl_create(8, 8, 1e-4, 1e-4, med)          # library-allocated workspace
    assert rc == 0
    assert P.fvnl_set_bc(h, 5, 0) == P.EARG
    assert P.fvnl_set_bc(h, 0, P.SOURCE, None) == P.EARG
    assert P.fvnl_set_bc(h, 0, P.PERIODIC) == 0
    assert P.fvnl_step(h, 1, 0.5, 1) == P.EARG              # lone PERIODIC side
    assert P.fvnl_set_bc(h, 1, P.PERIODIC) == 0
    assert P.fvnl_step(h, 1, -1.0, 1) == P.EARG
    assert P.fvnl_step(h, 1, 1.0, 0) == P.EARG              # fixed dt = 1 s: kappa far above 1/2
    assert P.fvnl_step(h, 3, 0.5, 1) == 0                   # equilibrium initial state steps cleanly
    rc, info = P.fvnl_get_info(h)
    assert rc == 0 and info["steps"] == 3 and abs(info["cfl"] - 0.5) < 1e-12
    assert P.fvnl_kernel_launches(h) > 0
    P.fvnl_destroy(h)
    ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    rc, h = P.fvnl_create(64, 64, 1e-4, 1e-4, med, workspace_ptr=(ws.data_ptr() + 255) // 256 * 256, workspace_bytes=512)
    assert rc == P.EALLOC
    assert "CFL" in P.fvnl_strerror(P.ECFL)


def _window_oracle_rect(w, q0, i0, j0, wx, wy, margin, steps, dt):
    """The oracle on a patch (window + margin on every side) cut out of the full periodic grid (modular gather); after
    `steps` steps with margin >= 3 steps + 3 the window cannot have seen the patch edge (dependency cone: 3 cells / step)."""
    from oracle.oracle import Oracle
    nxp, nyp = wx + 2 * margin, wy + 2 * margin
    ii = (np.arange(i0 - margin, i0 - margin + nxp) % w.nx)
    jj = (np.arange(j0 - margin, j0 - margin + nyp) % w.ny)
    it, jt = torch.as_tensor(ii, device=q0[0].device), torch.as_tensor(jj, device=q0[0].device)
    patch = [np.ascontiguousarray(q[jt][:, it].cpu().numpy()) for q in q0]
    o = Oracle(nxp, nyp, w.dx, w.dy, **w.medium, threads=0)
    for side in range(4):
        o.set_bc(side, 0)
    o.set_state(*patch)
    assert o.step(steps, dt, 0) == 0
    return [a[margin:margin + wy, margin:margin + wx] for a in o.get_state()], (ii[margin:margin + wx], jj[margin:margin + wy])


@pytest.mark.parametrize("n", [8192, 16384])
def test_c5_full_size_full_step_count_windows(n):
    """C5 at BASELINE.json's large sizes (8192^2, 16384^2) over its FULL step count (100), default kernel and launch
    configuration (what bench.py times).  The oracle cannot run the whole grid, so it recomputes windows of it cell by
    cell, each cut out with a margin (3 x 100 + 8 cells) wider than the dependency cone of the 100 steps: one on the
    periodic corner, one in the bulk, and one tall window (48 x 720 cells) placed on a seam between two strips of columns
    -- any chunk of rows of the automatic launch configuration shorter than 720 rows has a seam inside it.  Fixed dt: the
    CFL-mode dt depends on the whole grid, which only the CUDA path sees here (the dt control at full step count is
    covered by the whole-grid cases C2, C3, C5-2048 and C4).  Plus what holds at any size: sum of q conserved under
    periodic edges."""
    import paper_1311_3004_b200 as P
    w = W.c5_sweep(n=n)
    steps = w.steps
    assert steps == 100
    q0 = w.init(device="cuda")
    s = P.Solver(w.nx, w.ny, w.dx, w.dy, **w.medium)
    for side, (kind, src) in enumerate(w.bc):
        s.set_bc(side, kind, src)
    s.set_state(*q0)
    dt = w.value * w.dx / (w.medium["c0"] * 1.004)                  # nu = 0.9 / 1.004 x (max speed ~ 1.002): below nu_W
    sums0 = [float(q.sum(dtype=torch.float64)) for q in q0]
    assert s.step(steps, dt, 0) == 0
    assert 0.88 < s.info()["cfl"] < 0.9
    out = s.get_state()
    for m in range(3):
        assert abs(float(out[m].sum(dtype=torch.float64)) - sums0[m]) <= 1e-12 * w.cells ** 0.5 * max(1.0, abs(sums0[m]) / w.cells) * 50
    margin = 3 * steps + 8
    worst = 0.0
    for (i0, j0, wx, wy) in ((n - 24, n - 24, 48, 48), (n // 2 - 7, 3 * n // 4 + 11, 48, 48), (122 * 31 - 24, 377, 48, 720)):
        ref, (ii, jj) = _window_oracle_rect(w, q0, i0, j0, wx, wy, margin, steps, dt)
        got = [o_[torch.as_tensor(jj, device="cuda")][:, torch.as_tensor(ii, device="cuda")].cpu().numpy() for o_ in out]
        err = parity_error(got, ref)
        print(f"PARITY C5-{n} window ({i0},{j0}) {wx}x{wy} of {n}x{n} steps={steps} kernel=default err={err:.3e} tol={TOL:g}")
        worst = max(worst, err)
    assert worst <= TOL, f"C5-{n}: windowed parity error {worst:.3e}"


def test_c5_2048_full_size_full_step_count():
    """C5 at 2048^2 as BASELINE.json states it: the whole grid, 100 steps, nu_W = 0.9 in CFL mode, against the oracle."""
    check(W.c5_sweep(n=2048), cache_key="C5-2048")


@pytest.mark.parametrize("rows", [4, 7, 64, 1000])
@pytest.mark.parametrize("kernel", KERNELS[:2], ids=KIDS[:2])
def test_rows_per_block_choices(kernel, rows):
    """The one-pass kernels with forced chunk heights (down to chunks shorter than their own pipeline fill, and one
    chunk for the whole grid): chunk seams, ragged last chunk, periodic wrap inside the halo of the first chunk."""
    w = W.c3_random(n=300, ny=131, steps=25, sig_lo=3.0, sig_hi=12.0)
    check(w, kernel=kernel, rows_per_block=rows)
    w = W.c4_hifu(nx=260, ny=90, steps=40, focus_cells=60.0, aperture_cells=30.0, tau0=-1.0)
    check(w, kernel=kernel, rows_per_block=rows)


def test_c2_full_size():
    """C2 at BASELINE.json's full size and step count (1024^2, 500 steps, extrapolation edges, nu_W = 0.9): the oracle
    runs the whole problem (about half a minute on the box's cores); element-by-element parity plus the mirror symmetry
    of the centred pulse (P4) on the GPU result."""
    w = W.c2_pulse()
    err = check(w, cache_key="C2")
    assert err <= TOL
    s = solver_from_workload(w)
    assert s.step(w.steps, w.value, w.mode) == 0
    q1, q2, q3 = [a.cpu().numpy() for a in s.get_state()]
    # the oracle is mirror symmetric to round-off (pin P4); the CUDA path is within TOL of it, hence within 2 TOL of its
    # own mirror image
    amp = np.abs(q1 - 1.0).max()
    assert np.abs(q1 - q1[:, ::-1]).max() <= 2 * TOL * amp and np.abs(q1 - q1[::-1, :]).max() <= 2 * TOL * amp
    assert np.abs(q2 + q2[:, ::-1]).max() <= 2 * TOL * np.abs(q2).max()
    assert np.abs(q3 + q3[::-1, :]).max() <= 2 * TOL * np.abs(q3).max()


def test_c3_full_size_full_step_count():
    """C3 as BASELINE.json states it: the whole 4096^2 grid, periodic, 200 steps in CFL mode at nu_W = 0.8, element by
    element against the oracle (3.4 G cell-updates: a few minutes of the OpenMP oracle), plus conservation of sum q."""
    w = W.c3_random()
    q0 = [a.numpy() for a in w.init()]
    sums0 = [a.sum() for a in q0]
    gq, oq, gi, oi, fg, fo = run_both(w, cache_key="C3")
    assert fg == fo == 0 and gi["steps"] == oi["steps"] == 200
    for k in ("t", "dt", "M", "cfl"):
        assert gi[k] == pytest.approx(oi[k], rel=1e-12)
    assert abs(gi["cfl"] - w.value) < 1e-3
    for m in range(3):
        assert abs(gq[m].sum() - sums0[m]) <= 4e-8
    err = parity_error(gq, oq)
    print(f"PARITY C3 {w.nx}x{w.ny} steps=200 kernel=default err={err:.3e} tol={TOL:g}")
    assert err <= TOL


def test_c4_full_size_full_step_count():
    """C4 as BASELINE.json states it: 8192 x 2048, focused packet source, nu_W = 0.8 in CFL mode, 4000 steps, against the
    oracle's stored run of the WHOLE problem (tests/golden/c4_full_windows.txt, written by tests/golden/make_c4_windows.py:
    clock, whole-grid statistics and 20 x 20 windows after 400, 1000, 2000, 3000, 4000 steps).  Metric: SURVEY.md 8(d),
    per field max|Q_gpu - Q_orc| over the window / max|Q_orc - Q_eq| over the whole grid (stored by the oracle).

    What is asserted.  The north-star bar 1e-10 up to step 1000 AND after the full 4000 steps.  In between this problem
    amplifies ROUNDING differences between any two implementations of the scheme: the library's own three-pass kernels, run here beside
    the default kernel, are a second implementation that differs from it by rounding only, and the two drift apart by
    1e-9 .. 2e-8 by steps 2000-4000.  There the test asserts that the distance to the oracle is no larger than that
    measured distance between two correct implementations (and never above 1e-8), prints every number, and reports
    'ABOVE THE BAR' where 1e-10 is exceeded -- the bar is not claimed there."""
    import importlib.util
    import os
    spec = importlib.util.spec_from_file_location(
        "make_c4_windows", os.path.join(os.path.dirname(__file__), "golden", "make_c4_windows.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    if not os.path.exists(mod.OUT):
        pytest.skip("tests/golden/c4_full_windows.txt has not been generated (two hours of the oracle)")
    gold = mod.read()
    w = W.c4_hifu()
    assert (gold["config"]["nx"], gold["config"]["ny"], gold["config"]["nu_w"]) == (w.nx, w.ny, w.value)
    assert gold["config"]["steps"][-1] == w.steps == 4000
    import paper_1311_3004_b200 as P
    s = solver_from_workload(w, state=w.init(device="cuda"))
    s2 = solver_from_workload(w, state=w.init(device="cuda"))        # second implementation: the three-pass kernels
    s2.set_option(P.OPT_KERNEL, P.KERNEL_UNFUSED)
    win = gold["config"]["win"]
    done, report = 0, []
    sens = {}                                                            # the oracle against itself under FMA contraction
    sens_path = os.path.join(os.path.dirname(__file__), "golden", "c4_sensitivity.txt")   # (make_c4_sensitivity.py, oracle only)
    if os.path.exists(sens_path):
        for line in open(sens_path):
            if line.startswith("worst"):
                sens[int(line.split()[1])] = float(line.split()[2])
    have = [cp for cp in gold["config"]["steps"] if cp in gold["checkpoints"]]   # (a file copied from the script's .partial
    assert have and have == gold["config"]["steps"][:len(have)]                  # output holds the first checkpoints only)
    for cp in have:
        assert s.step(cp - done, w.value, w.mode) == 0
        assert s2.step(cp - done, w.value, w.mode) == 0
        done = cp
        ref = gold["checkpoints"][cp]
        info = s.info()
        assert info["steps"] == cp
        for k in ("t", "dt", "M", "cfl"):
            assert info[k] == pytest.approx(ref[k], rel=1e-11), (cp, k)
        out, out2 = s.get_state(), s2.get_state()
        drift = 0.0                                                     # default kernel vs three-pass kernels, whole grid
        for m in range(3):
            d = (out[m] - (1.0 if m == 0 else 0.0))
            st = ref["stats"][m]
            assert float(d.abs().max()) == pytest.approx(st["max"], rel=1e-8)
            assert abs(float(d.sum(dtype=torch.float64)) - st["sum"]) <= 1e-8 * st["l1"] + 1e-18
            assert float((d * d).sum(dtype=torch.float64)) == pytest.approx(st["l2"], rel=1e-8)
            drift = max(drift, float((out[m] - out2[m]).abs().max()) / st["max"])
        worst = 0.0
        for name, wd in ref["windows"].items():
            for m in range(3):
                got = out[m][wd["j0"]:wd["j0"] + win, wd["i0"]:wd["i0"] + win].cpu().numpy()
                err = np.abs(got - wd["q"][m]).max() / ref["stats"][m]["max"]
                print(f"PARITY C4-full step={cp} window={name}@({wd['i0']},{wd['j0']}) field=q{m + 1} err={err:.3e}")
                worst = max(worst, err)
        verdict = "within the bar" if worst <= TOL else "ABOVE THE BAR"
        print(f"PARITY C4 {w.nx}x{w.ny} step={cp} kernel=default err={worst:.3e} tol={TOL:g} {verdict}; "
              f"default vs three-pass kernels (rounding only) drift={drift:.3e}"
              + (f"; oracle vs oracle with FMA contraction (rounding only, same windows) {sens[cp]:.3e}" if cp in sens else ""))
        report.append((cp, worst, drift))
        if cp <= 1000 or cp == w.steps:                                   # ... and after the FULL step count (the north-star's bar)
            assert worst <= TOL, (cp, worst)
        else:
            assert worst <= min(max(TOL, drift), 1e-8), (cp, worst, drift)
    assert report[-1][0] == have[-1]
    if have[-1] != 4000:
        print(f"PARITY C4 golden file holds checkpoints up to step {have[-1]} only")


def test_c4_full_size_source_window():
    """C4 at full size (8192 x 2048, focused packet source on x-lo, nu_W = 0.8): 240 steps, by which the packet has entered
    (tau from -9.1 to -3.1 periods).  The oracle recomputes a patch that contains the source edge around the centre of
    the aperture, wide enough that the compared 64 x 64 cells at the edge cannot have seen the patch's other edges
    (3 cells per step); fixed dt so that both take the same steps."""
    import paper_1311_3004_b200 as P
    from oracle.oracle import Oracle
    w = W.c4_hifu()
    steps, size = 240, 64
    margin = 3 * steps + 8
    s = solver_from_workload(w, state=w.init(device="cuda"))
    dt = 0.8 * w.dx / (w.medium["c0"] * 1.003)
    assert s.step(steps, dt, 0) == 0
    out = s.get_state()
    jc = w.ny // 2
    j_lo = max(0, jc - size // 2 - margin)
    j_hi = min(w.ny, jc + size // 2 + margin)
    nyp, nxp = j_hi - j_lo, size + margin
    o = Oracle(nxp, nyp, w.dx, w.dy, **w.medium, threads=0)
    src = dict(w.bc[0][1])
    src["centre_m"] = src["centre_m"] - j_lo * w.dy                 # the aperture in the patch's own y coordinate
    o.set_bc(0, P.SOURCE, src)
    for side in (1, 2, 3):
        o.set_bc(side, P.EXTRAP)
    o.set_state(np.ones((nyp, nxp)), np.zeros((nyp, nxp)), np.zeros((nyp, nxp)))
    assert o.step(steps, dt, 0) == 0
    ref = [a[jc - size // 2 - j_lo: jc + size // 2 - j_lo, :size] for a in o.get_state()]
    got = [a[jc - size // 2: jc + size // 2, :size].cpu().numpy() for a in out]
    assert np.abs(ref[0] - 1.0).max() > 1e-5                           # the packet is there
    err = parity_error(got, ref)
    print(f"PARITY C4 source window {w.nx}x{w.ny} steps={steps} kernel=default err={err:.3e} tol={TOL:g}")
    assert err <= TOL


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_extreme_aspect_ratios(kernel):
    """One very long row of strips (100 003 x 4) and one very tall strip (4 x 20 011): many strips with a ragged last one,
    a grid narrower than a strip's halo, many chunks."""
    import paper_1311_3004_b200 as P
    for nx, ny in ((100003, 4), (4, 20011)):
        for bc in (P.PERIODIC, P.EXTRAP):
            w = W.c3_random(n=nx, ny=ny, steps=12, sig_lo=2.0, sig_hi=6.0, seed=99 + nx)
            w.bc = [(bc, None)] * 4
            check(w, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_equilibrium_is_a_fixed_point(kernel):
    """The degenerate case: Q = Q_eq stays Q_eq bit for bit under every passive edge kind (all waves vanish identically),
    M = 1/dx exactly (|s| = 1 at rest), and zero steps change nothing."""
    import paper_1311_3004_b200 as P
    for bc in (P.PERIODIC, P.EXTRAP, P.REFLECT):
        s = P.Solver(150, 37, 1e-4, 1e-4, c0=1500.0, rho0=1000.0, beta=3.5, delta=4.3e-6)
        select(s, kernel)
        for side in range(4):
            s.set_bc(side, bc)
        assert s.step(0, 0.9, 1) == 0
        assert s.step(25, 0.9, 1) == 0
        q1, q2, q3 = s.get_state()
        assert torch.equal(q1, torch.ones_like(q1)) and not q2.any() and not q3.any()
        info = s.info()
        assert info["steps"] == 25 and info["M"] == pytest.approx(1.0 / 1e-4, rel=1e-15) and info["cfl"] == pytest.approx(0.9, rel=1e-14)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_sources_on_every_side(kernel):
    """Focused packet on x-hi, plane piston on y-lo, continuous focused source on y-hi, Taylor profile on x-lo (each with
    extrapolation or reflection elsewhere): the side-dependent signs of (43b,c) and all four blocks of the boundary
    kernel's buffer."""
    import paper_1311_3004_b200 as P
    dx = W.LAMBDA_1MHZ / 32
    base = dict(shape=P.PACKET, amp=4e-4, freq_hz=1e6, focus_m=50 * dx, centre_m=70 * dx, half_aperture_m=30 * dx,
                t0_s=-1.5e-6, steep=0.0)
    cases = []
    w = W.c2_pulse(n=180, ny=140, sigma_cells=5.0, steps=120, amp=2e-4)
    w.bc = [(P.EXTRAP, None), (P.SOURCE, dict(base)), (P.REFLECT, None), (P.EXTRAP, None)]
    cases.append(w)
    w = W.c2_pulse(n=150, ny=170, sigma_cells=5.0, steps=120, amp=2e-4)
    w.bc = [(P.EXTRAP, None), (P.EXTRAP, None), (P.SOURCE, dict(base, shape=P.SINE, focus_m=0.0, half_aperture_m=0.0, t0_s=0.0)),
            (P.SOURCE, dict(base, shape=P.SINE, t0_s=0.0, centre_m=80 * dx))]
    cases.append(w)
    for w in cases:
        check(w, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_oblique_taylor_shocks(kernel):
    """the profile (41) propagating at theta_T = pi/8 and pi/4 on a 2-D grid, analytic cells
    (41) on all four sides (both sweeps, the splitting and every edge kernel path at once).  Perturbation 1e-7 on a unit
    background: bar 1e-7 on one scale for all fields, as for C1-T."""
    import math
    for theta in (math.pi / 8, math.pi / 4):
        w = W.c1t_taylor(eta=10, nu_w=0.9, x_lo=-4.0, x_hi=10.0, y_lo=-5.0, y_hi=8.0, theta=theta)
        check(w, steps=90, tol=1e-7, metric=parity_error_global, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS, ids=KIDS)
def test_moving_domain(kernel):
    """the domain moves with the wave (fvnl_shift).  (a) a pulse under extrapolation
    edges, the domain moved by 1..3 cells every few steps; (b) the Taylor test with analytic cells (41) entering on the
    right, moved one cell whenever the front has advanced by one, as the oracle's driver does."""
    w = W.c2_pulse(n=260, ny=90, sigma_cells=6.0, steps=1, amp=1e-3)
    state = [a.numpy().copy() for a in w.init()]
    o = oracle_from_workload(w, threads=0, state=state)
    s = solver_from_workload(w, state=[torch.from_numpy(a) for a in state])
    select(s, kernel)
    for n, k in ((7, 1), (5, 3), (11, 2), (4, 0), (9, 1)):
        assert o.step(n, 0.9, 1) == 0 and s.step(n, 0.9, 1) == 0
        o.shift(k)
        s.shift(k)
    assert o.step(6, 0.9, 1) == 0 and s.step(6, 0.9, 1) == 0
    assert s.info()["t"] == pytest.approx(o.info()["t"], rel=1e-12)
    err = parity_error([a.cpu().numpy() for a in s.get_state()], o.get_state())
    print(f"PARITY moving pulse kernel={kernel} err={err:.3e}")
    assert err <= TOL
    tw = W.c1t_taylor(eta=10, nu_w=0.9, x_lo=-6.0, x_hi=6.0, ny=6, y_periodic=False)
    state = [a.numpy().copy() for a in tw.init()]
    o = oracle_from_workload(tw, threads=0, state=state)
    s = solver_from_workload(tw, state=[torch.from_numpy(a) for a in state])
    select(s, kernel)
    shifted = 0
    for _ in range(120):
        assert o.step(1, 0.9, 1) == 0 and s.step(1, 0.9, 1) == 0
        k = int(np.floor(o.info()["t"] * 10)) - shifted
        if k > 0:
            o.shift(k)
            s.shift(k)
            shifted += k
    assert shifted >= 100
    err = parity_error_global([a.cpu().numpy() for a in s.get_state()], o.get_state())
    print(f"PARITY moving Taylor kernel={kernel} shifted={shifted} err={err:.3e}")
    assert err <= 1e-7
    import paper_1311_3004_b200 as P
    with pytest.raises(P.FvnlError):
        solver_from_workload(W.c3_random(n=16, ny=16)).shift(1)
