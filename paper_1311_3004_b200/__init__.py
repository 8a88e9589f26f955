"""paper_1311_3004_b200 -- thin Python binding of libfvnl.so (include/fvnl.h).

The per-time-step 2-D high-resolution finite-volume update of arXiv 1311.3004 (Sections II-III), fp64, one B200.
Argument marshalling only: every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch provides
device memory and the stream.  There is no CPU fallback: without the built library or without a CUDA device
this module raises.

    s = Solver(nx, ny, dx, dy, c0=1500., rho0=1000., beta=3.5, delta=4.3e-6)
    s.set_bc(XLO, SOURCE, dict(shape=SINE, amp=1/1500., freq_hz=1e6)); ...
    s.set_state(q1, q2, q3)            # torch tensors, CUDA or CPU, float64, (ny, nx)
    flags = s.step(100, 0.9, mode=1)   # 100 steps at nu_W = 0.9
    q1, q2, q3 = s.get_state()

The module-level fvnl_* functions are the C entry points with the same names and argument order.
"""
import ctypes as C
import os

import torch

from . import build as _build

EXTRAP, PERIODIC, REFLECT, SOURCE = 0, 1, 2, 3
SINE, PACKET, TANH = 0, 1, 2
XLO, XHI, YLO, YHI = 0, 1, 2, 3
OK, EARG, EALLOC, ECUDA, ESTATE, ESIZE = 0, 1, 2, 3, 4, 5
NOALLOC_MAX_BYTES = 16 << 20
ECFL, ENONREAL, ENONPOS, ENAN = 16, 32, 64, 128
OPT_KERNEL, OPT_ROWS_PER_BLOCK, OPT_KERNEL_TIMING, OPT_VARIANT, OPT_SMALL_GRID = 0, 1, 2, 3, 4
TIMED_STEP, TIMED_XSWEEP, TIMED_YSWEEP, TIMED_SOURCE = 0, 1, 2, 3
KERNEL_DEFAULT, KERNEL_UNFUSED = 0, 1
ON_HOST, ON_DEVICE, PLANES_F64 = 0, 1, 2


class fvnl_medium(C.Structure):
    _fields_ = [("c0", C.c_double), ("rho0", C.c_double), ("beta", C.c_double), ("delta", C.c_double)]


class fvnl_source(C.Structure):
    _fields_ = [("shape", C.c_int), ("amp", C.c_double), ("freq_hz", C.c_double), ("focus_m", C.c_double),
                ("centre_m", C.c_double), ("half_aperture_m", C.c_double), ("t0_s", C.c_double),
                ("steep", C.c_double), ("theta", C.c_double)]


class FvnlError(RuntimeError):
    def __init__(self, where, code):
        self.code = code
        super().__init__(f"{where}: {fvnl_strerror(code)} ({code})")


_lib = None
_vp = C.c_void_p


def lib():
    """Load libfvnl.so (built in-tree by paper_1311_3004_b200.build; a missing compiler or library is an error)."""
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build(force=bool(os.environ.get("FVNL_REBUILD"))))   # mtime-gated: never a stale binary
        L.fvnl_workspace_bytes.restype = C.c_size_t
        L.fvnl_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int]
        L.fvnl_create.argtypes = [C.POINTER(_vp), C.c_int, C.c_int, C.c_double, C.c_double, C.POINTER(fvnl_medium),
                                  C.c_int, _vp, _vp, C.c_size_t]
        L.fvnl_destroy.restype = None
        L.fvnl_destroy.argtypes = [_vp]
        L.fvnl_set_bc.argtypes = [_vp, C.c_int, C.c_int, C.POINTER(fvnl_source)]
        L.fvnl_set_option.argtypes = [_vp, C.c_int, C.c_int]
        L.fvnl_set_state.argtypes = [_vp, _vp, _vp, _vp, C.c_int]
        L.fvnl_set_clock.argtypes = [_vp, C.c_double, C.c_double]
        L.fvnl_shift.argtypes = [_vp, C.c_int]
        L.fvnl_step.argtypes = [_vp, C.c_long, C.c_double, C.c_int]
        L.fvnl_get_state.argtypes = [_vp, _vp, _vp, _vp, C.c_int]
        L.fvnl_get_info.argtypes = [_vp] + [C.POINTER(C.c_double)] * 4 + [C.POINTER(C.c_long)]
        L.fvnl_get_kernel_time.argtypes = [_vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_long)]
        L.fvnl_probe_fp64.argtypes = [_vp, C.POINTER(C.c_double)]
        L.fvnl_kernel_launches.restype = C.c_long
        L.fvnl_kernel_launches.argtypes = [_vp]
        L.fvnl_step_noalloc.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.POINTER(fvnl_medium), C.POINTER(C.c_int),
                                        C.POINTER(C.POINTER(fvnl_source)), C.c_double, C.c_double] + [_vp] * 8
        L.fvnl_strerror.restype = C.c_char_p
        L.fvnl_strerror.argtypes = [C.c_int]
        _lib = L
    return _lib


# ---- the C entry points, same names, same order ----------------------------------------------------------------
def fvnl_workspace_bytes(nx, ny, precision=64):
    return lib().fvnl_workspace_bytes(nx, ny, precision)


def fvnl_create(nx, ny, dx, dy, medium, precision=64, cuda_stream=0, workspace_ptr=0, workspace_bytes=0):
    h = _vp()
    rc = lib().fvnl_create(C.byref(h), nx, ny, dx, dy, C.byref(medium), precision, _vp(cuda_stream or None),
                           _vp(workspace_ptr or None), workspace_bytes)
    return rc, h


def fvnl_destroy(h):
    lib().fvnl_destroy(h)


def fvnl_set_bc(h, side, kind, src=None):
    return lib().fvnl_set_bc(h, side, kind, C.byref(src) if src is not None else None)


def fvnl_set_option(h, option, value):
    return lib().fvnl_set_option(h, option, value)


def fvnl_set_state(h, p1, p2, p3, where):
    return lib().fvnl_set_state(h, _vp(p1), _vp(p2), _vp(p3), int(where))


def fvnl_shift(h, cells):
    return lib().fvnl_shift(h, int(cells))


def fvnl_set_clock(h, t_s, last_M):
    return lib().fvnl_set_clock(h, t_s, last_M)


def fvnl_step(h, nsteps, value, mode):
    return lib().fvnl_step(h, int(nsteps), float(value), int(mode))


def fvnl_get_state(h, p1, p2, p3, where):
    return lib().fvnl_get_state(h, _vp(p1), _vp(p2), _vp(p3), int(where))


def fvnl_get_info(h):
    t, dt, cfl, M = C.c_double(), C.c_double(), C.c_double(), C.c_double()
    n = C.c_long()
    rc = lib().fvnl_get_info(h, C.byref(t), C.byref(dt), C.byref(cfl), C.byref(M), C.byref(n))
    return rc, dict(t=t.value, dt=dt.value, cfl=cfl.value, M=M.value, steps=n.value)


def fvnl_get_kernel_time(h, which):
    ms, n = C.c_double(), C.c_long()
    rc = lib().fvnl_get_kernel_time(h, int(which), C.byref(ms), C.byref(n))
    return rc, ms.value, n.value


def fvnl_probe_fp64(cuda_stream=0):
    v = C.c_double()
    rc = lib().fvnl_probe_fp64(_vp(cuda_stream or None), C.byref(v))
    return rc, v.value


def fvnl_kernel_launches(h):
    return lib().fvnl_kernel_launches(h)


def fvnl_step_noalloc(nx, ny, dx, dy, medium, bc_kind, bc_source, t, dt, q_in, q_out, flags_ptr=0, cuda_stream=0):
    """One fixed-dt step with no allocation (include/fvnl.h).  bc_kind: four ints; bc_source: four fvnl_source or None;
    q_in / q_out: three DEVICE pointers (ints) each; flags_ptr: device pointer to one int, or 0."""
    kinds = (C.c_int * 4)(*bc_kind)
    srcs = (C.POINTER(fvnl_source) * 4)()
    keep = []
    for k, s in enumerate(bc_source or (None,) * 4):
        if s is not None:
            keep.append(s)
            srcs[k] = C.pointer(s)
    return lib().fvnl_step_noalloc(nx, ny, dx, dy, C.byref(medium), kinds, srcs, t, dt, *[_vp(p) for p in q_in],
                                   *[_vp(p) for p in q_out], _vp(flags_ptr or None), _vp(cuda_stream or None))


def fvnl_strerror(code):
    return lib().fvnl_strerror(int(code)).decode()


# ---- convenience object -----------------------------------------------------------------------------------------
class Solver:
    """One fvnl context on the current CUDA device and torch's current stream.

    precision 64: state tensors are (ny, nx) float64 holding q.  precision 32 (perturbation form, include/fvnl.h): the
    context stores float32 planes (rho' = q1 - 1, q2, q3); set_state / get_state take either such float32 tensors, or
    float64 tensors holding the standard q, which the LIBRARY converts on the device (FVNL_PLANES_F64)."""

    def __init__(self, nx, ny, dx, dy, c0, rho0, beta, delta, device="cuda", stream=None, precision=64):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1311_3004_b200 needs a CUDA device; there is no CPU fallback")
        self.device = torch.device(device)
        if self.device.type != "cuda":
            raise RuntimeError("paper_1311_3004_b200 runs on CUDA devices only")
        self.nx, self.ny = int(nx), int(ny)
        self.precision = int(precision)
        self.dtype = torch.float64 if self.precision == 64 else torch.float32
        self._h = None
        with torch.cuda.device(self.device):
            nbytes = fvnl_workspace_bytes(self.nx, self.ny, self.precision)
            if nbytes == 0:
                raise FvnlError("fvnl_workspace_bytes", EARG)
            # torch owns the device memory; +256 so that a 256-byte aligned base always exists
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._ws.data_ptr() + 255) // 256 * 256
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            rc, h = fvnl_create(self.nx, self.ny, dx, dy, fvnl_medium(c0, rho0, beta, delta), self.precision,
                                self._stream.cuda_stream, base, nbytes)
        if rc:
            raise FvnlError("fvnl_create", rc)
        self._h = h

    def close(self):
        if self._h:
            fvnl_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, where, rc):
        if rc:
            raise FvnlError(where, rc)

    def set_bc(self, side, kind, src=None):
        s = None
        if src is not None:
            s = src if isinstance(src, fvnl_source) else fvnl_source(**src)
        self._check("fvnl_set_bc", fvnl_set_bc(self._h, side, kind, s))

    def set_option(self, option, value):
        self._check("fvnl_set_option", fvnl_set_option(self._h, option, value))

    def _prep(self, a):
        a = torch.as_tensor(a)
        if a.dtype not in (torch.float64, self.dtype) or a.numel() != self.nx * self.ny:
            raise ValueError("state planes must be float64 (q) or the context's own dtype, with nx*ny elements")
        return a.contiguous()

    def set_state(self, q1, q2, q3):
        """Copy a state in; CUDA tensors are read on the device, CPU tensors / arrays from host memory."""
        q = [self._prep(a) for a in (q1, q2, q3)]
        on_dev = q[0].is_cuda
        if any(a.is_cuda != on_dev or a.dtype != q[0].dtype for a in q):
            raise ValueError("all three planes must live on the same side and have one dtype")
        where = ON_DEVICE if on_dev else ON_HOST
        if self.precision == 32 and q[0].dtype == torch.float64:      # standard q for an fp32 context: the library converts,
            q = [a.to(self.device) for a in q]                         # on the device (torch only moves the bytes there)
            where = ON_DEVICE | PLANES_F64
        with torch.cuda.device(self.device):
            self._check("fvnl_set_state", fvnl_set_state(self._h, q[0].data_ptr(), q[1].data_ptr(), q[2].data_ptr(), where))
            if where & PLANES_F64:
                self._stream.synchronize()                             # the temporaries above are read asynchronously

    def shift(self, cells):
        """Move the domain by `cells` cells in +x (second stage of PAPER.md:287)."""
        self._check("fvnl_shift", fvnl_shift(self._h, cells))

    def set_clock(self, t, last_M=0.0):
        self._check("fvnl_set_clock", fvnl_set_clock(self._h, t, last_M))

    def step(self, nsteps, value, mode):
        """mode 0: value = dt [s]; mode 1: value = nu_W.  Returns the sticky device flag word (0 = clean)."""
        with torch.cuda.device(self.device):
            rc = fvnl_step(self._h, nsteps, value, mode)
        if 0 < rc < 16:
            raise FvnlError("fvnl_step", rc)
        return rc

    def get_state(self, out=None, host=False, as_q64=False):
        """Current state as three (ny, nx) tensors in the context's own form: on the device, or (host=True) in (pinned)
        host memory.  as_q64 (fp32 contexts): float64 device tensors holding the standard q, converted by the library.
        `out`: three preallocated tensors to fill instead."""
        if out is None:
            if as_q64:
                out = [torch.empty(self.ny, self.nx, dtype=torch.float64, device=self.device) for _ in range(3)]
            elif host:
                out = [torch.empty(self.ny, self.nx, dtype=self.dtype, pin_memory=True) for _ in range(3)]
            else:
                out = [torch.empty(self.ny, self.nx, dtype=self.dtype, device=self.device) for _ in range(3)]
        where = ON_DEVICE if out[0].is_cuda else ON_HOST
        if self.precision == 32 and out[0].dtype == torch.float64:
            if not out[0].is_cuda:
                raise ValueError("float64 output of an fp32 context is produced on the device")
            where |= PLANES_F64
        elif out[0].dtype != self.dtype:
            raise ValueError("output planes must have the context's dtype")
        with torch.cuda.device(self.device):
            self._check("fvnl_get_state", fvnl_get_state(self._h, out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), where))
        return out

    def info(self):
        rc, d = fvnl_get_info(self._h)
        self._check("fvnl_get_info", rc)
        return d

    def kernel_time(self, which):
        """(summed device ms, launches) of one timed kernel since the last read (needs OPT_KERNEL_TIMING = 1)."""
        rc, ms, n = fvnl_get_kernel_time(self._h, which)
        self._check("fvnl_get_kernel_time", rc)
        return ms, n

    def kernel_launches(self):
        return fvnl_kernel_launches(self._h)
