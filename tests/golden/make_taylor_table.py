"""Writes tests/golden/taylor_table_oracle.txt: the oracle's errors on the paper's Taylor-shock test, theta_T = 0.

Calls ONLY oracle/ (and the input generators in workloads/); never the CUDA path.  Takes ~10 min on 4 cores, which
is why the table is stored; tests/test_oracle_pins.py re-runs the cheap rows live and checks the stored ones against
the numbers the paper prints in Table I.

Set-up (readings A11, A12, A15 in DESIGN.md): 1-D-in-2-D grid, ny = 4, x in [-15, 115], dx = 1/eta,
initial state (41) at t = 0 sampled at cell centres, x-sides Dirichlet (41) at t_n, y-sides periodic, K = 1e-7,
lagged CFL control nu_W, run until the first t_n >= 100 - dt/2; E_k of (42) on q1 - 1 over |x - t| <= 5.

    python tests/golden/make_taylor_table.py
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.oracle import Oracle  # noqa: E402
import workloads as W  # noqa: E402

ETAS = (5, 10, 20, 41, 82)
NUS = (0.6, 0.7, 0.8, 0.9, 0.99)


def taylor_errors(eta, nu, threads=0, y_periodic=True):
    w = W.c1t_taylor(eta=eta, nu_w=nu, y_periodic=y_periodic)
    o = Oracle(w.nx, w.ny, w.dx, w.dy, **w.medium, threads=threads)
    for s, (k, src) in enumerate(w.bc):
        o.set_bc(s, k, src)
    o.set_state(*[a.numpy() for a in w.init()])
    t_end = w.extra["t_end"]
    o.step(max(int(t_end * eta / nu) - 8, 1), nu, 1)
    cfls = []
    while o.info()["t"] < t_end - 0.5 * o.info()["dt"]:
        flags = o.step(1, nu, 1)
        cfls.append(o.info()["cfl"])
    info = o.info()
    assert flags == 0
    q1 = o.get_state()[0][1]
    x = (np.arange(w.nx) + 0.5) * w.dx + w.extra["x_lo"]
    ref = W.taylor_reference(torch.from_numpy(x), info["t"], w.extra["K"]).numpy() - 1.0
    m = np.abs(x - info["t"]) <= 5.0
    err = np.abs((q1 - 1.0) - ref)[m]
    E1 = err.sum() / np.abs(ref)[m].sum()
    Einf = err.max() / np.abs(ref)[m].max()
    return E1, Einf, info


THETAS = (0.0, np.pi / 32, np.pi / 16, np.pi / 8, np.pi / 4)
OBLIQUE_ETAS = (5, 10, 20)


def taylor_errors_oblique(eta, nu, theta, T=12.0, lo=-8.0, hi=22.0, half_width=2.0, threads=0):
    """Table I rows theta_T != 0 at a size the CPU oracle can run: the profile (41) under the
    standard rotation on the square [lo, hi]^2, analytic cells (41) on all four sides, run from t = 0 to
    the first t_n >= T - dt/2.  E_k of (42) on q1 - 1 over the cells within 5 units of the front along the propagation
    direction (reading A12) and within `half_width` units of the ray through the origin across it -- the paper's 10-unit
    line, as a strip of cells.  (The paper's eta = 82, t = 100 rows need ~1e12 cell-updates: out of the oracle's reach.)"""
    w = W.c1t_taylor(eta=eta, nu_w=nu, t_end=T, x_lo=lo, x_hi=hi, y_lo=lo, y_hi=hi, theta=theta)
    o = Oracle(w.nx, w.ny, w.dx, w.dy, **w.medium, threads=threads)
    for s, (k, src) in enumerate(w.bc):
        o.set_bc(s, k, src)
    o.set_state(*[a.numpy() for a in w.init()])
    o.step(max(int(T * eta / nu) - 4, 1), nu, 1)
    flags = 0
    while o.info()["t"] < T - 0.5 * o.info()["dt"]:
        flags |= o.step(1, nu, 1)
    assert flags == 0
    info = o.info()
    q1 = o.get_state()[0]
    x = (np.arange(w.nx) + 0.5) * w.dx + lo
    y = (np.arange(w.ny) + 0.5) * w.dy + lo
    X, Y = np.meshgrid(x, y)
    ct, st = np.cos(theta), np.sin(theta)
    xi, perp = X * ct + Y * st, -X * st + Y * ct
    ref = W.taylor_reference(torch.from_numpy(xi), info["t"], w.extra["K"]).numpy() - 1.0
    m = (np.abs(xi - info["t"]) <= 5.0) & (np.abs(perp) <= half_width)
    err = np.abs((q1 - 1.0) - ref)[m]
    return err.sum() / np.abs(ref)[m].sum(), err.max() / np.abs(ref)[m].max(), info


def taylor_errors_moving(eta, nu, t_end=100.0, half_length=15.0, threads=0):
    """The two-stage technique of PAPER.md:281-287 on the theta_T = 0 test: the domain [-half_length, half_length] stays
    still until the front (at x = t) reaches its centre -- here from the start -- and then moves with it, one cell each
    time the front has advanced by one cell; analytic cells (41) on all sides "for both stages"."""
    w = W.c1t_taylor(eta=eta, nu_w=nu, t_end=t_end, x_lo=-half_length, x_hi=half_length, y_periodic=True)
    o = Oracle(w.nx, w.ny, w.dx, w.dy, **w.medium, threads=threads)
    for s, (k, src) in enumerate(w.bc):
        o.set_bc(s, k, src)
    o.set_state(*[a.numpy() for a in w.init()])
    shifted = 0
    flags = 0
    while o.info()["t"] < t_end - 0.5 * o.info()["dt"]:
        flags |= o.step(1, nu, 1)
        k = int(np.floor(o.info()["t"] * eta)) - shifted          # cells the front has advanced since the last move
        if k > 0:
            o.shift(k)
            shifted += k
    assert flags == 0
    info = o.info()
    q1 = o.get_state()[0][1]
    x = (np.arange(w.nx) + 0.5) * w.dx - half_length + shifted * w.dx
    ref = W.taylor_reference(torch.from_numpy(x), info["t"], w.extra["K"]).numpy() - 1.0
    m = np.abs(x - info["t"]) <= 5.0
    err = np.abs((q1 - 1.0) - ref)[m]
    return err.sum() / np.abs(ref)[m].sum(), err.max() / np.abs(ref)[m].max(), info, shifted


def write_oblique_table():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "taylor_oblique_oracle.txt")
    lines = ["# written by tests/golden/make_taylor_table.py --oblique (oracle only).  Taylor profile (41) at an angle theta_T on",
             "# [-8, 22]^2, nu_W = 0.9, t = 12 (taylor_errors_oblique).  columns: eta theta_T E1 Einf t_final steps"]
    for eta in OBLIQUE_ETAS:
        for th in THETAS:
            E1, Einf, info = taylor_errors_oblique(eta, 0.9, th)
            lines.append(f"{eta} {th!r} {E1:.6e} {Einf:.6e} {info['t']:.12f} {info['steps']}")
            print(lines[-1], flush=True)
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    if "--oblique" in sys.argv:
        write_oblique_table()
        sys.exit(0)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "taylor_table_oracle.txt")
    lines = ["# written by tests/golden/make_taylor_table.py (oracle only). columns: eta nu_W E1 Einf t_final steps last_cfl"]
    for eta in ETAS:
        for nu in NUS:
            E1, Einf, info = taylor_errors(eta, nu)
            lines.append(f"{eta} {nu} {E1:.6e} {Einf:.6e} {info['t']:.12f} {info['steps']} {info['cfl']:.12f}")
            print(lines[-1], flush=True)
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")
