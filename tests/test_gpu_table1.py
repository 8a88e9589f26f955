"""The paper's Taylor-shock test at the paper's own resolution and time (Table I: eta = 82 cells across the
shock, t = 100 shock widths) -- with the CUDA path as the instrument, against what the PAPER prints.

The CPU oracle reaches eta = 82 only for theta_T = 0 (a 1-D-in-2-D grid; tests/test_oracle_pins.py, P1); the oblique rows need
~1e11 ... 1e12 cell-updates each, seconds on a B200.  Nothing here compares with the oracle: the expected values are the
paper's (tests/golden/paper_table1.txt, with citations).  What the paper fixes and what it leaves open:

  * fixed: the profile (41) with its standard rotation, analytic cells (41) on all four sides, K = 1e-7,
    nu_W in {0.6 ... 0.99}, the error norms (42) over a 10-unit line, eta = 82, t = 100;
  * open: the size of the (moving) domain and where the 10-unit line lies in it.  The analytic cells around the domain feed the
    exact solution in, so the error measured near an edge is smaller than in the open: the printed oblique errors are
    reproduced in order of magnitude and in their ORDER (they grow with theta_T), not digit by digit -- with the front 13
    units from the nearest edge the CUDA path measures E1 = 2.1e-4 ... 2.9e-4 where the paper prints 2.7e-4 ... 1.3e-3.

Asserted: (a) theta_T = 0, for nu_W = 0.6, 0.9, 0.99: E1 and E_inf inside the printed [best, worst] interval of the eta = 82
columns (+- 30 %, the acceptance of the oracle's pin P1); (b) every angle: E1 < 0.3 % and E_inf < 2 % ("reaching, when eta = 82, values below 0.3 % for E1, and below 2 % for
E_inf") and not above the printed worst value (x 1.3); (c) both norms grow with theta_T, as every printed column
does; (d) at theta_T = pi/32, the angle nearest to the aligned case, E1 is within a factor 2 of the printed best value.
"""
import math
import os

import pytest
import torch

import workloads as W
from helpers import solver_from_workload

pytestmark = pytest.mark.gpu

ETA, T_END, MARGIN = 82, 100.0, 8.0


def paper_rows():
    """{theta label: dict(E1=(best, worst), Einf=(best, worst))} from tests/golden/paper_table1.txt (worst may be None)."""
    rows = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_table1.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            th, norm, best, worst = line.split()
            rows.setdefault(th, {})[norm] = (float(best), None if worst == "-" else float(worst))
    return rows


def taylor_errors_gpu(theta, nu):
    """E1, E_inf of (42) on q1 - 1 at t = 100: cells within 5 units of the front along the propagation direction and within 2
    units of the ray through the origin across it (reading A12b of DESIGN.md), static domain with the front 13 units from the
    nearest edge at the end."""
    ct, st = math.cos(theta), math.sin(theta)
    if theta:
        lo = -MARGIN
        w = W.c1t_taylor(eta=ETA, nu_w=nu, t_end=T_END, x_lo=lo, x_hi=T_END * ct + MARGIN + 5.0, y_lo=lo,
                         y_hi=T_END * st + MARGIN + 5.0, theta=theta)
        ylo = lo
    else:
        lo, ylo = -15.0, 0.0
        w = W.c1t_taylor(eta=ETA, nu_w=nu, t_end=T_END, x_lo=lo, x_hi=115.0, y_periodic=True)
    s = solver_from_workload(w, state=w.init(device="cuda"))
    flags = s.step(max(int(T_END * ETA / nu) - 8, 1), nu, 1)
    while s.info()["t"] < T_END - 0.5 * s.info()["dt"]:
        flags |= s.step(1, nu, 1)
    assert flags == 0
    info = s.info()
    q1 = s.get_state()[0]
    x = (torch.arange(w.nx, dtype=torch.float64, device="cuda") + 0.5) * w.dx + lo
    y = (torch.arange(w.ny, dtype=torch.float64, device="cuda") + 0.5) * w.dy + ylo
    xi = x[None, :] * ct + y[:, None] * st
    ref = W.taylor_reference(xi, info["t"], w.extra["K"]) - 1.0
    m = (xi - info["t"]).abs() <= 5.0
    if theta:
        m = m & ((-x[None, :] * st + y[:, None] * ct).abs() <= 2.0)
    err = ((q1 - 1.0) - ref).abs()[m]
    return float(err.sum() / ref.abs()[m].sum()), float(err.max() / ref.abs()[m].max()), info, (w.nx, w.ny)


def test_table1_theta0_row_on_the_gpu():
    p = paper_rows()["0"]
    for nu in (0.6, 0.9, 0.99):
        E1, Einf, info, grid = taylor_errors_gpu(0.0, nu)
        print(f"TABLE1 theta_T=0 eta={ETA} nu_W={nu} grid={grid[0]}x{grid[1]} steps={info['steps']} E1={E1:.3e} "
              f"(paper {p['E1'][0]:.2e} .. {p['E1'][1]:.2e}) Einf={Einf:.3e} (paper {p['Einf'][0]:.2e} .. {p['Einf'][1]:.2e})")
        assert p["E1"][0] * 0.7 <= E1 <= p["E1"][1] * 1.3                     # the acceptance of the oracle's pin P1
        assert p["Einf"][0] * 0.7 <= Einf <= p["Einf"][1] * 1.3


def test_table1_oblique_rows_on_the_gpu():
    rows = paper_rows()
    out = []
    for label, theta in (("pi/32", math.pi / 32), ("pi/16", math.pi / 16), ("pi/8", math.pi / 8), ("pi/4", math.pi / 4)):
        E1, Einf, info, grid = taylor_errors_gpu(theta, 0.9)
        p = rows[label]
        print(f"TABLE1 theta_T={label} eta={ETA} nu_W=0.9 grid={grid[0]}x{grid[1]} steps={info['steps']} E1={E1:.3e} "
              f"(paper best {p['E1'][0]:.2e}, worst {p['E1'][1]}) Einf={Einf:.3e} (paper best {p['Einf'][0]:.2e}, worst {p['Einf'][1]})")
        assert E1 < 3e-3 and Einf < 2e-2                                    # (b) PAPER.md:372
        assert E1 <= 1.3 * (p["E1"][1] or p["E1"][0]) and Einf <= 1.3 * (p["Einf"][1] or p["Einf"][0])
        out.append((E1, Einf))
    for a, b in zip(out, out[1:]):                                          # (c) every printed column grows with theta_T
        assert b[0] > a[0] and b[1] > a[1]
    assert 0.5 * rows["pi/32"]["E1"][0] <= out[0][0] <= 2.0 * rows["pi/32"]["E1"][0]   # (d)
