"""Shared test helpers: build an oracle / a CUDA context from a workloads.Workload, and the parity metric."""
import numpy as np


def oracle_from_workload(w, threads=0, state=None):
    from oracle.oracle import Oracle
    o = Oracle(w.nx, w.ny, w.dx, w.dy, **w.medium, threads=threads)
    for side, (kind, src) in enumerate(w.bc):
        o.set_bc(side, kind, src)
    if state is None:
        state = [a.numpy() for a in w.init()]
    o.set_state(*state)
    return o


def solver_from_workload(w, state=None, device="cuda", precision=64):
    import torch
    from paper_1311_3004_b200 import Solver
    s = Solver(w.nx, w.ny, w.dx, w.dy, **w.medium, device=device, precision=precision)
    for side, (kind, src) in enumerate(w.bc):
        s.set_bc(side, kind, src)
    if state is None:
        state = w.init()
    s.set_state(*[torch.as_tensor(a) for a in state])
    return s


def parity_error_global(gpu, orc):
    """max_m max|Q_gpu - Q_orc| / max_m max|Q_orc - Q_eq|: one scale for all fields.  Used only where a field is pure
    round-off noise in the oracle itself (C1-T with analytic y-edges: q3 ~ 1e-11 next to a 1e-7 perturbation on a
    unit background), so that the per-field ratio would compare round-off with round-off."""
    diff = pert = 0.0
    for m, (g, o) in enumerate(zip(gpu, orc)):
        g = np.asarray(g, dtype=np.float64)
        o = np.asarray(o, dtype=np.float64)
        assert np.isfinite(g).all(), f"field {m}: non-finite values on the GPU"
        pert = max(pert, np.abs(o - (1.0 if m == 0 else 0.0)).max())
        diff = max(diff, np.abs(g - o).max())
    return diff / pert


def parity_error(gpu, orc):
    """SURVEY.md 8(d) parity metric: per field m, E^m = max|Q_gpu - Q_orc| / max|Q_orc - Q_eq|, Q_eq = (1,0,0).
    A field that is identically zero in the oracle must be identically zero on the GPU.  Returns max_m E^m."""
    worst = 0.0
    for m, (g, o) in enumerate(zip(gpu, orc)):
        g = np.asarray(g, dtype=np.float64)
        o = np.asarray(o, dtype=np.float64)
        assert g.shape == o.shape
        assert np.isfinite(g).all(), f"field {m}: non-finite values on the GPU"
        pert = np.abs(o - (1.0 if m == 0 else 0.0)).max()
        diff = np.abs(g - o).max()
        if pert == 0.0:
            assert diff == 0.0, f"field {m} is identically at equilibrium in the oracle but not on the GPU ({diff})"
            continue
        worst = max(worst, diff / pert)
    return worst
