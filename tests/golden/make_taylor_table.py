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


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "taylor_table_oracle.txt")
    lines = ["# written by tests/golden/make_taylor_table.py (oracle only). columns: eta nu_W E1 Einf t_final steps last_cfl"]
    for eta in ETAS:
        for nu in NUS:
            E1, Einf, info = taylor_errors(eta, nu)
            lines.append(f"{eta} {nu} {E1:.6e} {Einf:.6e} {info['t']:.12f} {info['steps']} {info['cfl']:.12f}")
            print(lines[-1], flush=True)
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")
