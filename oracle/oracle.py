"""ctypes wrapper of oracle/fvnl_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only; all arithmetic is in the C++ file.  Imports nothing from paper_1311_3004_b200.
"""
import ctypes as C

import numpy as np

from . import build as _build

EXTRAP, PERIODIC, REFLECT, SOURCE = 0, 1, 2, 3
SINE, PACKET, TANH = 0, 1, 2
XLO, XHI, YLO, YHI = 0, 1, 2, 3
ECFL, ENONREAL, ENONPOS, ENAN = 16, 32, 64, 128


class _Medium(C.Structure):
    _fields_ = [("c0", C.c_double), ("rho0", C.c_double), ("beta", C.c_double), ("delta", C.c_double)]


class OrcSource(C.Structure):
    _fields_ = [("shape", C.c_int), ("amp", C.c_double), ("freq_hz", C.c_double), ("focus_m", C.c_double),
                ("centre_m", C.c_double), ("half_aperture_m", C.c_double), ("t0_s", C.c_double),
                ("steep", C.c_double), ("theta", C.c_double)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.POINTER(_Medium)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_set_bc.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(OrcSource)]
        L.orc_set_state.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.orc_get_state.argtypes = [C.c_void_p, _dp, _dp, _dp]
        L.orc_set_clock.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_get_info.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, C.POINTER(C.c_long)]
        L.orc_step.argtypes = [C.c_void_p, C.c_long, C.c_double, C.c_int]
        L.orc_step_stages.argtypes = [C.c_void_p, C.c_long, C.c_double, C.c_int, C.c_int]
        L.orc_flux.argtypes = [_dp, C.c_double, C.c_int, _dp]
        L.orc_riemann.argtypes = [_dp, _dp, C.c_double, _dp, _dp, _dp, _dp]
        L.orc_mc_phi.restype = C.c_double
        L.orc_mc_phi.argtypes = [C.c_double]
        L.orc_sweep_line.argtypes = [C.c_int, _dp, C.c_double, C.c_double, _dp, _dp]
        L.orc_source_cell.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, _dp]
        L.orc_shift.argtypes = [C.c_void_p, C.c_int]
        L.orc_prepass.restype = C.c_double
        L.orc_prepass.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _arr(x):
    return np.ascontiguousarray(x, dtype=np.float64)


class Oracle:
    """One simulation context of the CPU oracle.  State arrays are (ny, nx) float64, x fastest."""

    def __init__(self, nx, ny, dx, dy, c0, rho0, beta, delta, threads=1):
        self.nx, self.ny = int(nx), int(ny)
        m = _Medium(c0, rho0, beta, delta)
        self._h = lib().orc_create(self.nx, self.ny, dx, dy, C.byref(m))
        if not self._h:
            raise ValueError("orc_create: bad arguments")
        self.threads = lib().orc_set_threads(self._h, threads)

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def set_bc(self, side, kind, src=None):
        s = None
        if src is not None:
            s = src if isinstance(src, OrcSource) else OrcSource(**src)
        rc = lib().orc_set_bc(self._h, side, kind, C.byref(s) if s is not None else None)
        if rc:
            raise ValueError(f"orc_set_bc -> {rc}")

    def set_state(self, q1, q2, q3):
        q1, q2, q3 = _arr(q1), _arr(q2), _arr(q3)
        assert q1.size == q2.size == q3.size == self.nx * self.ny
        lib().orc_set_state(self._h, _p(q1), _p(q2), _p(q3))

    def get_state(self):
        out = [np.empty((self.ny, self.nx), dtype=np.float64) for _ in range(3)]
        lib().orc_get_state(self._h, _p(out[0]), _p(out[1]), _p(out[2]))
        return out

    def set_clock(self, t, last_M=0.0):
        lib().orc_set_clock(self._h, t, last_M)

    def info(self):
        t, dt, cfl, M = C.c_double(), C.c_double(), C.c_double(), C.c_double()
        n = C.c_long()
        lib().orc_get_info(self._h, C.byref(t), C.byref(dt), C.byref(cfl), C.byref(M), C.byref(n))
        return dict(t=t.value, dt=dt.value, cfl=cfl.value, M=M.value, steps=n.value)

    def step(self, nsteps, value, mode, stages=7):
        """mode 0: value = dt [s]; mode 1: value = nu_W.  Returns the sticky flag word."""
        return lib().orc_step_stages(self._h, int(nsteps), float(value), int(mode), int(stages))

    def prepass(self):
        return lib().orc_prepass(self._h)

    def source_cell(self, side, along_m, xc_m, t, yc_m=0.0):
        out = np.zeros(3)
        inside = lib().orc_source_cell(self._h, side, along_m, xc_m, yc_m, t, _p(out))
        return bool(inside), out

    def shift(self, cells):
        """Move the domain by `cells` cells in +x (second stage of PAPER.md:287)."""
        rc = lib().orc_shift(self._h, int(cells))
        if rc:
            raise ValueError(f"orc_shift -> {rc}")


def flux(q, beta, direction):
    q = _arr(q)
    f = np.zeros(3)
    lib().orc_flux(_p(q), beta, direction, _p(f))
    return f


def riemann(QL, QR, beta):
    QL, QR = _arr(QL), _arr(QR)
    s, W, am, ap = np.zeros(3), np.zeros(9), np.zeros(3), np.zeros(3)
    flag = lib().orc_riemann(_p(QL), _p(QR), beta, _p(s), _p(W), _p(am), _p(ap))
    return dict(s=s, W=W.reshape(3, 3), amdq=am, apdq=ap, flag=flag)


def mc_phi(theta):
    return lib().orc_mc_phi(float(theta))


def sweep_line(cells, lam, beta):
    """cells: (n+4, 3) with 2 ghosts each side -> (out (n,3), smax, flag)."""
    cells = _arr(cells)
    n = cells.shape[0] - 4
    out = np.zeros((n, 3))
    sm = C.c_double()
    flag = lib().orc_sweep_line(n, _p(cells), lam, beta, _p(out), C.byref(sm))
    return out, sm.value, flag
