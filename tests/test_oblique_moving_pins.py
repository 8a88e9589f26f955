"""Pins of the oracle for the two 'next' rows that touch its arithmetic: oblique Taylor shocks (Table I rows
theta_T != 0) and the moving domain of the second stage.

What can and cannot be pinned.  The paper prints, for theta_T != 0, worst convergence rates over eta = 5..82 and errors at
eta = 82, t = 100.  One such run is ~1e12 cell-updates (a 2-D domain of ~1e8 cells over ~1.4e4 steps): out of reach of the
CPU oracle (1e7 cell-updates/s), and the paper does not state its domain.  What the paper fixes and a small run can check:
  * the construction itself -- "a standard rotation change of variables" of (41): theta_T = pi/2 must be the
    theta_T = 0 run with x and y (and q2 and q3) exchanged, EXACTLY, and theta_T = pi its mirror image;
  * the order of the Table I rows: both printed error columns grow monotonically with theta_T from 0 to pi/4 ("errors
    diminish when the propagation is aligned with the mesh"), the oblique rates are lower than the aligned
    one and all are above one;
  * a rotated field that is NOT a travelling solution (a wrong sign or exchanged sine / cosine anywhere in the rotation)
    does not stay within a factor ~2 of the aligned error.
The stored table tests/golden/taylor_oblique_oracle.txt is written by tests/golden/make_taylor_table.py --oblique (oracle
only); the cheap rows are re-run live here.
"""
import importlib.util
import math
import os

import numpy as np
import pytest

import workloads as W
from oracle.oracle import Oracle, EXTRAP, PERIODIC, SOURCE, XLO, XHI, YLO, YHI, TANH
from helpers import oracle_from_workload

HERE = os.path.dirname(os.path.abspath(__file__))


def _script():
    spec = importlib.util.spec_from_file_location("make_taylor_table", os.path.join(HERE, "golden", "make_taylor_table.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def _oblique_table():
    rows = {}
    with open(os.path.join(HERE, "golden", "taylor_oblique_oracle.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            eta, th, e1, einf, *_ = line.split()
            rows[(int(eta), round(float(th), 6))] = (float(e1), float(einf))
    return rows


THETAS = [0.0, math.pi / 32, math.pi / 16, math.pi / 8, math.pi / 4]


def test_table1_rows_are_ordered_as_the_paper_prints_them():
    """E1 at eta = 82 = 2.36e-05 < 2.70e-04 < 4.62e-04 < 7.97e-04 < 1.31e-03 and E_inf = 2.96e-04 <
    3.56e-03 < 6.73e-03 < 1.06e-02 < 1.12e-02 for theta_T = 0 < pi/32 < pi/16 < pi/8 < pi/4.  The oracle's errors at
    eta = 5, 10, 20 grow in the same order, the growth gets stronger as the mesh is refined (the aligned error falls
    faster: PAPER.md:349-352 worst rates 1.15-1.28 against 1.63), and every rate is above one."""
    paper = {"E1": [2.36e-05, 2.70e-04, 4.62e-04, 7.97e-04, 1.31e-03], "Einf": [2.96e-04, 3.56e-03, 6.73e-03, 1.06e-02, 1.12e-02]}
    for col in paper.values():
        assert all(a < b for a, b in zip(col, col[1:]))
    rows = _oblique_table()
    for eta in (5, 10, 20):
        for col in (0, 1):
            errs = [rows[(eta, round(th, 6))][col] for th in THETAS]
            assert all(a < b for a, b in zip(errs, errs[1:])), (eta, col, errs)
            assert errs[-1] < 2.0 * errs[0]                           # still a travelling solution at every angle
    growth = [rows[(eta, round(math.pi / 4, 6))][0] / rows[(eta, 0.0)][0] for eta in (5, 10, 20)]
    assert growth[0] < growth[1] < growth[2]
    for th in THETAS:
        e = [rows[(eta, round(th, 6))][0] for eta in (5, 10, 20)]
        rate = -np.polyfit(np.log([5.0, 10.0, 20.0]), np.log(e), 1)[0]
        assert 1.0 < rate < 2.2, (th, rate)
        if th > 0:
            e0 = [rows[(eta, 0.0)][0] for eta in (5, 10, 20)]
            assert rate < -np.polyfit(np.log([5.0, 10.0, 20.0]), np.log(e0), 1)[0]


def test_oblique_table_is_what_the_oracle_computes():
    mod = _script()
    rows = _oblique_table()
    for eta, th in ((5, 0.0), (5, math.pi / 8), (5, math.pi / 4), (10, math.pi / 16)):
        E1, Einf, info = mod.taylor_errors_oblique(eta, 0.9, th)
        assert E1 == pytest.approx(rows[(eta, round(th, 6))][0], rel=2e-6)
        assert Einf == pytest.approx(rows[(eta, round(th, 6))][1], rel=2e-6)
        assert abs(info["cfl"] - 0.9) < 1e-6


def _run(w, steps, nu=0.9):
    o = oracle_from_workload(w)
    assert o.step(steps, nu, 1) == 0
    return o.get_state(), o.info()


def test_rotation_by_a_right_angle_and_by_pi_is_exact():
    """The rotated set-up at theta_T = pi/2 is the aligned one with the axes (and q2, q3) exchanged: for a field that does
    not vary across the propagation direction the other sweep is an exact no-op, so the two runs agree to round-off
    (cos(pi/2) = 6e-17 and sin(pi) = 1e-16 are not zero: 1e-10 of the perturbation is allowed, any slip in the rotation
    is of the order of the perturbation itself).  theta_T = pi is the mirror image in x.
    Fails under: sine and cosine exchanged in the profile or in the velocity, a wrong sign of either, y measured from a
    wrong origin in the y-ghost rows."""
    eta, n_long, n_short = 8, 30, 4
    # (periodic across the propagation direction: with analytic cells there the edge rows see the numerical error of the
    # interior against the exact ghost values, which the X-then-Y splitting treats differently in x and in y, reading A9)
    a = W.c1t_taylor(eta=eta, x_lo=-15.0, x_hi=15.0, ny=n_short, y_periodic=True)                  # along x
    b = W.c1t_taylor(eta=eta, x_lo=0.0, x_hi=n_short / eta, y_lo=-15.0, y_hi=15.0, theta=math.pi / 2)   # along y
    b.bc[0] = b.bc[1] = (PERIODIC, None)
    assert (b.nx, b.ny) == (a.ny, a.nx)
    qa, ia = _run(a, 60)
    qb, ib = _run(b, 60)
    assert ia["t"] == pytest.approx(ib["t"], rel=1e-12)
    K = 1e-7
    assert np.abs(qa[0] - qb[0].T).max() <= 1e-10 * K
    assert np.abs(qa[1] - qb[2].T).max() <= 1e-10 * K
    assert np.abs(qa[2]).max() == 0.0 and np.abs(qb[1]).max() <= 1e-10 * K
    assert np.abs(qa[0] - 1).max() > 0.9 * K
    # theta = pi: the front moves in -x; mirror image of the aligned run about the domain centre
    c = W.c1t_taylor(eta=eta, x_lo=-15.0, x_hi=15.0, ny=n_short, theta=math.pi, y_periodic=True)
    qc, ic = _run(c, 60)
    assert ic["t"] == pytest.approx(ia["t"], rel=1e-12)
    assert np.abs(qc[0] - qa[0][:, ::-1]).max() <= 1e-10 * K
    assert np.abs(qc[1] + qa[1][:, ::-1]).max() <= 1e-10 * K


def test_oblique_source_cells_are_the_rotated_field():
    """(41) under the rotation, at single cells: the value depends on position only through x cos + y sin, the velocity is
    parallel to the propagation direction and has the size of the density perturbation -- on every side and in the corners."""
    th = 0.3
    w = W.c1t_taylor(eta=10, x_lo=-3.0, x_hi=9.0, y_lo=-2.0, y_hi=6.0, theta=th)
    o = oracle_from_workload(w)
    ct, st = math.cos(th), math.sin(th)
    t = 1.7
    for side in (XLO, XHI, YLO, YHI):
        for (xe, ye) in ((-0.15, 3.05), (12.05, -0.25), (4.45, 8.15), (2.0, 2.0)):
            inside, q = o.source_cell(side, ye if side < 2 else xe, xe, t, yc_m=ye)
            xi = (xe - 3.0) * ct + (ye - 2.0) * st
            assert inside and q[0] == pytest.approx(1 - 1e-7 * math.tanh(W.TAYLOR_STEEP * (xi - t)), abs=3e-16)
            assert q[1] * st - q[2] * ct == pytest.approx(0.0, abs=1e-22)
            assert math.hypot(q[1], q[2]) == pytest.approx(abs(q[0] - 1.0), rel=1e-12, abs=1e-22)
            # a second point on the same phase line gives the same cell
            _, q2 = o.source_cell(side, (ye + 0.5 * ct) if side < 2 else (xe - 0.5 * st), xe - 0.5 * st, t, yc_m=ye + 0.5 * ct)
            assert q2[0] == pytest.approx(q[0], abs=3e-16)


# ------------------------------------------------------------------------------------------------- moving domain
def test_shift_commutes_with_the_scheme():
    """"in the second stage the domain moves with the propagation wave".  Moving the domain re-indexes the
    cells; the scheme is translation invariant, so advancing n steps and then moving by k cells equals moving first and
    advancing afterwards, bit for bit, wherever neither edge can have been felt (3 cells per step)."""
    w = W.c2_pulse(n=96, ny=40, sigma_cells=4.0, steps=1, amp=2e-3)
    dt = 0.8 * w.dx / w.medium["c0"]
    a = oracle_from_workload(w)
    assert a.step(6, dt, 0) == 0
    a.shift(5)
    b = oracle_from_workload(w)
    b.shift(5)
    assert b.step(6, dt, 0) == 0
    qa, qb = a.get_state(), b.get_state()
    lo, hi = 3 * 6 + 2, 96 - 5 - 3 * 6 - 2
    for m in range(3):
        assert np.array_equal(qa[m][:, lo:hi], qb[m][:, lo:hi])
    # re-indexing: column i now holds what column i + 5 held; the entering columns copy the last one (extrapolation)
    c = oracle_from_workload(w)
    q0 = c.get_state()
    c.shift(7)
    q1 = c.get_state()
    for m in range(3):
        assert np.array_equal(q1[m][:, :89], q0[m][:, 7:])
        assert np.array_equal(q1[m][:, 89:], np.repeat(q0[m][:, -1:], 7, axis=1))
    with pytest.raises(ValueError):
        oracle_from_workload(W.c3_random(n=16, ny=16)).shift(1)            # periodic in x: nothing to move into
    # analytic x-hi edge: the entering columns are the profile (41) at their OWN centres, and the frame moves along, so
    # that a second move continues where the first one ended
    tw = W.c1t_taylor(eta=10, x_lo=-3.0, x_hi=0.5, ny=4, y_periodic=True)     # (x-hi edge inside the front: cells differ)
    o = oracle_from_workload(tw)
    o.shift(7)
    o.shift(3)
    x = (np.arange(tw.nx) + 0.5) * tw.dx - 3.0 + 10 * tw.dx
    ref = 1.0 - 1e-7 * np.tanh(W.TAYLOR_STEEP * x)
    q = o.get_state()
    assert np.abs(q[0][1] - ref).max() <= 3e-16 and np.abs(q[1][1] - (ref - 1.0)).max() <= 3e-16
    assert np.abs(np.diff(ref[-12:])).min() > 0.0                          # (the entering cells are not copies of one another)


def test_moving_domain_reproduces_the_static_taylor_run():
    """The paper ran its Taylor test with the two-stage technique ((41) on all borders "for both stages").
    A 30-unit domain that moves with the front gives the errors of the static 130-unit domain of the stored Table I run."""
    mod = _script()
    rows = {}
    with open(os.path.join(HERE, "golden", "taylor_table_oracle.txt")) as f:
        for line in f:
            if not line.startswith("#") and line.strip():
                eta, nu, e1, einf, *_ = line.split()
                rows[(int(eta), float(nu))] = (float(e1), float(einf))
    for eta, nu in ((5, 0.9), (10, 0.8)):
        E1, Einf, info, shifted = mod.taylor_errors_moving(eta, nu)
        assert shifted >= 100 * eta - 1 and info["t"] >= 100.0 - info["dt"]
        assert E1 == pytest.approx(rows[(eta, nu)][0], rel=0.02)
        assert Einf == pytest.approx(rows[(eta, nu)][1], rel=0.02)
