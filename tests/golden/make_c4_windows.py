"""Writes tests/golden/c4_full_windows.txt: the oracle's state of BASELINE.json's config C4 at FULL size and FULL step count.

Calls ONLY oracle/ (and the input generators in workloads/); never the CUDA path.  C4 = 8192 x 2048 cells, focused
packet source (43a-d) on x-lo, extrapolation elsewhere, nu_W = 0.8, 4000 steps in CFL mode
(lagged dt control): 67 G cell-updates, about two hours of the OpenMP oracle on 8 cores -- too long
for pytest, which is why the result is stored.  Because the dependency cone of 4000 steps (3 cells per step) is larger
than the grid, no sub-domain reproduces the final state: the oracle runs the WHOLE problem and this script keeps

  * at each checkpoint (steps 400 -- packet being emitted --, 1000, 2000, 3000 -- packet at the focus --, 4000) the
    clock (t, dt, M, nu) and, per field, max|Q - Q_eq| over the whole grid (the denominator of the parity metric of
    SURVEY.md 8(d)), sum(Q - Q_eq), sum|Q - Q_eq| and sum (Q - Q_eq)^2 over the whole grid;
  * WIN x WIN windows of the state, every value as a C99 hex float (exact): on the source edge at the centre of the
    aperture and half-way to its rim, at the geometric focus, around the cell where |q1 - 1| is largest and around the
    cell where |q3| is largest (off axis).

tests/test_gpu_parity.py::test_c4_full_size_full_step_count advances the CUDA path over the same 4000 steps and compares
element by element.  tests/test_oracle_pins.py re-runs this script on a scaled-down C4 so that the file format and the
script cannot go stale.

    python tests/golden/make_c4_windows.py [--threads N]            # writes tests/golden/c4_full_windows.txt
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.oracle import Oracle  # noqa: E402
import workloads as W  # noqa: E402

WIN = 20
CHECKPOINTS = (400, 1000, 2000, 3000, 4000)
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c4_full_windows.txt")


def clamp_origin(c, n, win):
    """Origin of a window of `win` cells centred on cell c, kept inside [0, n)."""
    return int(min(max(c - win // 2, 0), n - win))


def window_list(w, q, win):
    """[(name, i0, j0)]: fixed windows (source edge, focus) and data-dependent ones (extrema of the oracle's state)."""
    nx, ny = w.nx, w.ny
    jc = ny // 2
    out = [("edge_axis", 0, clamp_origin(jc, ny, win)),
           ("edge_half_aperture", 0, clamp_origin(jc + int(w.extra["aperture_cells"] / 2), ny, win)),
           ("focus", clamp_origin(int(w.extra["focus_cells"]), nx, win), clamp_origin(jc, ny, win))]
    j, i = np.unravel_index(np.argmax(np.abs(q[0] - 1.0)), q[0].shape)
    out.append(("peak_q1", clamp_origin(i, nx, win), clamp_origin(j, ny, win)))
    j, i = np.unravel_index(np.argmax(np.abs(q[2])), q[2].shape)
    out.append(("peak_q3", clamp_origin(i, nx, win), clamp_origin(j, ny, win)))
    return out


def hexrow(a):
    return " ".join(float(x).hex() for x in a)


def run(w, checkpoints, win, threads, log=None, partial=None):
    """Advance the oracle over the workload in CFL mode, returning the lines of the golden file."""
    o = Oracle(w.nx, w.ny, w.dx, w.dy, **w.medium, threads=threads)
    for s, (k, src) in enumerate(w.bc):
        o.set_bc(s, k, src)
    o.set_state(*[a.numpy() for a in w.init()])
    lines = [f"config {w.name} {w.nx} {w.ny} {w.value!r} {win} " + " ".join(str(c) for c in checkpoints)]
    done = 0
    t0 = time.time()
    for cp in checkpoints:
        flags = o.step(cp - done, w.value, w.mode)
        done = cp
        assert flags == 0, f"oracle flags {flags} at step {cp}"
        info = o.info()
        assert info["steps"] == cp
        q = o.get_state()
        lines.append(f"checkpoint {cp} {info['t'].hex()} {info['dt'].hex()} {info['M'].hex()} {info['cfl'].hex()}")
        for m in range(3):
            d = q[m] - (1.0 if m == 0 else 0.0)
            lines.append(f"stat {cp} {m} {float(np.abs(d).max()).hex()} {float(d.sum()).hex()} "
                         f"{float(np.abs(d).sum()).hex()} {float((d * d).sum()).hex()}")
        for name, i0, j0 in window_list(w, q, win):
            lines.append(f"window {cp} {name} {i0} {j0}")
            for m in range(3):
                for j in range(j0, j0 + win):
                    lines.append(f"row {cp} {name} {m} {j} " + hexrow(q[m][j, i0:i0 + win]))
        if partial:                                  # a two-hour run: keep what is done so far
            with open(partial, "w") as f:
                f.write(HEADER + "\n".join(lines) + "\n")
        if log:
            log(f"step {cp}: t = {info['t']:.6e} s, nu = {info['cfl']:.6f}, max|q1-1| = {np.abs(q[0] - 1).max():.3e}, "
                f"{time.time() - t0:.0f} s")
    return lines


HEADER = """# written by tests/golden/make_c4_windows.py (oracle only; never the CUDA path).  C4 of BASELINE.json at full size.
# config <name> <nx> <ny> <nu_W> <window size> <checkpoint steps ...>
# checkpoint <step> <t [s]> <last dt [s]> <last M [1/m]> <last nu>                               (C99 hex floats)
# stat <step> <field m> <max|Q-Qeq|> <sum(Q-Qeq)> <sum|Q-Qeq|> <sum(Q-Qeq)^2>                   (whole grid)
# window <step> <name> <i0> <j0>  then  row <step> <name> <field m> <j> <values of cells i0 .. i0+win-1>
"""


def read(path=OUT):
    """Parse a file written by this script -> dict(config=..., checkpoints={step: dict(clock, stats, windows)})."""
    out = {"checkpoints": {}}
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            if k == "config":
                out["config"] = dict(name=v[0], nx=int(v[1]), ny=int(v[2]), nu_w=float(v[3]), win=int(v[4]),
                                     steps=[int(x) for x in v[5:]])
            elif k == "checkpoint":
                t, dt, M, cfl = (float.fromhex(x) for x in v[1:5])
                out["checkpoints"][int(v[0])] = dict(t=t, dt=dt, M=M, cfl=cfl, stats={}, windows={})
            elif k == "stat":
                mx, sm, l1, l2 = (float.fromhex(x) for x in v[2:6])
                out["checkpoints"][int(v[0])]["stats"][int(v[1])] = dict(max=mx, sum=sm, l1=l1, l2=l2)
            elif k == "window":
                win = out["config"]["win"]
                out["checkpoints"][int(v[0])]["windows"][v[1]] = dict(i0=int(v[2]), j0=int(v[3]),
                                                                    q=np.full((3, win, win), np.nan))
            elif k == "row":
                wd = out["checkpoints"][int(v[0])]["windows"][v[1]]
                wd["q"][int(v[2]), int(v[3]) - wd["j0"], :] = [float.fromhex(x) for x in v[4:]]
    return out


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--out", default=OUT)
    args = ap.parse_args(argv)
    w = W.c4_hifu()
    lines = run(w, CHECKPOINTS, WIN, args.threads, log=lambda s: print(s, flush=True),
                partial=args.out + ".partial")
    tmp = args.out + ".tmp"
    with open(tmp, "w") as f:
        f.write(HEADER + "\n".join(lines) + "\n")
    os.replace(tmp, args.out)
    if os.path.exists(args.out + ".partial"):
        os.remove(args.out + ".partial")
    print("wrote", args.out)


if __name__ == "__main__":
    main()
