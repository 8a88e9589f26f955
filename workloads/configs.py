"""The synthetic workloads of BASELINE.json / SURVEY.md 8(d), each scalable down to a test size.

Every factory returns a `Workload`: a pure description (grid, medium, four boundary descriptors, time-step mode,
step count) plus `init(device)` that draws the initial state.  State = the paper's dimensionless q of (22)
(PAPER.md:133), three (ny, nx) float64 tensors, x fastest.

Boundary descriptor: (kind, source) with kind in EXTRAP/PERIODIC/REFLECT/SOURCE and `source` a dict with the
fields of `fvnl_source` (include/fvnl.h).  Side order: x-lo, x-hi, y-lo, y-hi.
"""
import math
from dataclasses import dataclass, field
from typing import Callable, Dict, List, Optional, Tuple

import torch

from .rng import splitmix64_uniform

EXTRAP, PERIODIC, REFLECT, SOURCE = 0, 1, 2, 3
SINE, PACKET, TANH = 0, 1, 2

# water, BASELINE.json configs: c0 = 1500 m/s, rho0 = 1000 kg/m^3, beta = 3.5, diffusivity 4.3e-6 m^2/s
MEDIUM_WATER = dict(c0=1500.0, rho0=1000.0, beta=3.5, delta=4.3e-6)
LAMBDA_1MHZ = 1500.0 / 1.0e6          # 1.5 mm

# reading A11: L of (20) is the 10 %-90 % distance of the tanh profile -> tanh(c (x - t)), c = 2 atanh(0.8)
TAYLOR_STEEP = 2.0 * math.atanh(0.8)


def _src(shape, amp, freq_hz=0.0, focus_m=0.0, centre_m=0.0, half_aperture_m=0.0, t0_s=0.0, steep=0.0, theta=0.0):
    return dict(shape=shape, amp=amp, freq_hz=freq_hz, focus_m=focus_m, centre_m=centre_m,
                half_aperture_m=half_aperture_m, t0_s=t0_s, steep=steep, theta=theta)


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    dx: float
    dy: float
    medium: Dict[str, float]
    bc: List[Tuple[int, Optional[dict]]]
    mode: int                 # 0: value = dt [s]; 1: value = nu_W
    value: float
    steps: int
    init: Callable[..., Tuple[torch.Tensor, torch.Tensor, torch.Tensor]]
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return self.nx * self.ny


def _equilibrium(nx, ny):
    def init(device="cpu"):
        return (torch.ones(ny, nx, dtype=torch.float64, device=device),
                torch.zeros(ny, nx, dtype=torch.float64, device=device),
                torch.zeros(ny, nx, dtype=torch.float64, device=device))
    return init


# ---------------------------------------------------------------------------------------------------------------
def c1_piston(nx=512, ny=4, steps=2000, cells_per_lambda=64, u0=1.0, nu_w=0.9) -> Workload:
    """C1: plane piston, sinusoidal velocity 1 MHz, amplitude u0 at x = 0 (plane-wave limit of (43))."""
    med = dict(MEDIUM_WATER)
    dx = LAMBDA_1MHZ / cells_per_lambda
    src = _src(SINE, amp=u0 / med["c0"], freq_hz=1.0e6)
    return Workload("C1", nx, ny, dx, dx, med, [(SOURCE, src), (EXTRAP, None), (PERIODIC, None), (PERIODIC, None)],
                    1, nu_w, steps, _equilibrium(nx, ny), "plane piston, q3 == 0 exactly")


def taylor_reference(x, t, K=1.0e-7, steep=TAYLOR_STEEP):
    """(41) with reading A11: q1 = 1 - K tanh(steep (x - t)), dimensionless x, t."""
    return 1.0 - K * torch.tanh(steep * (x - t))


def c1t_taylor(eta=20, nu_w=0.9, t_end=100.0, ny=4, x_lo=-15.0, x_hi=115.0, K=1.0e-7, beta=3.5,
               y_periodic=False, theta=0.0, y_lo=0.0, y_hi=None) -> Workload:
    """C1-T: the paper's own Taylor-shock test.  Dimensionless: c0 = rho0 = 1, dx = 1/eta,
    delta~ = K beta / steep (the Taylor balance for tanh(steep (x-t)) of amplitude K).
    theta = theta_T, the propagation angle from the x_1 axis: the profile (41) under the standard rotation,
    q1 = 1 - K tanh(steep (x cos(theta) + y sin(theta) - t)), (q2, q3) = (q1 - 1)(cos(theta), sin(theta)), on a 2-D grid
    x in [x_lo, x_hi], y in [y_lo, y_hi] (y_hi = None: ny rows), analytic cells (41) on all four sides."""
    nx = int(round((x_hi - x_lo) * eta))
    dx = 1.0 / eta
    if y_hi is not None:
        ny = int(round((y_hi - y_lo) * eta))
    med = dict(c0=1.0, rho0=1.0, beta=beta, delta=K * beta / TAYLOR_STEEP)
    ct, st = math.cos(theta), math.sin(theta)
    # x, y of fvnl_source TANH are measured from the x-lo / y-lo edge: xi_phys = xi_edge + (x_lo ct + y_lo st) -> t0
    src = _src(TANH, amp=K, t0_s=-(x_lo * ct + y_lo * st), steep=TAYLOR_STEEP, theta=theta)
    ysides = (PERIODIC, None) if y_periodic else (SOURCE, dict(src))

    def init(device="cpu"):
        x = (torch.arange(nx, dtype=torch.float64, device=device) + 0.5) * dx + x_lo
        y = (torch.arange(ny, dtype=torch.float64, device=device) + 0.5) * dx + y_lo
        xi = x[None, :] * ct + y[:, None] * st
        q1 = taylor_reference(xi, 0.0, K).contiguous()
        return q1, (q1 - 1.0) * ct, (q1 - 1.0) * st + 0.0

    return Workload(f"C1-T(eta={eta},nu={nu_w},theta={theta:.4f})" if theta else f"C1-T(eta={eta},nu={nu_w})", nx, ny, dx, dx, med,
                    [(SOURCE, dict(src)), (SOURCE, dict(src)), ysides, ysides], 1, nu_w, 0, init,
                    "run until t >= t_end", extra=dict(t_end=t_end, x_lo=x_lo, y_lo=y_lo, K=K, eta=eta, theta=theta))


def c2_pulse(n=1024, steps=500, sigma_cells=20.0, amp=1.0e-3, nu_w=0.9, ny=None) -> Workload:
    """C2: centred Gaussian density pulse, zero velocity, extrapolation edges."""
    nx, ny = n, (n if ny is None else ny)
    dx = LAMBDA_1MHZ / 32

    def init(device="cpu"):
        i = torch.arange(nx, dtype=torch.float64, device=device) - (nx - 1) / 2.0
        j = torch.arange(ny, dtype=torch.float64, device=device) - (ny - 1) / 2.0
        r2 = j[:, None] ** 2 + i[None, :] ** 2
        q1 = 1.0 + amp * torch.exp(-r2 / (2.0 * sigma_cells ** 2))
        return q1, torch.zeros_like(q1), torch.zeros_like(q1)

    return Workload("C2", nx, ny, dx, dx, dict(MEDIUM_WATER), [(EXTRAP, None)] * 4, 1, nu_w, steps, init,
                    "state is L2 resident at 1024^2")


def _multi_gaussian(nx, ny, seed, n_gauss=32, amp=5.0e-4, sig_lo=5.0, sig_hi=50.0, vel=0.1, c0=1500.0,
                    rows_per_chunk=1024):
    """32 seeded Gaussians (periodic minimum-image distance) + i.i.d. U[-vel,vel] m/s velocities (reading A24)."""
    def init(device="cpu"):
        u = splitmix64_uniform(seed, 0, 4 * n_gauss, device=device).reshape(n_gauss, 4)
        amps = (2.0 * u[:, 0] - 1.0) * amp
        sigs = sig_lo + (sig_hi - sig_lo) * u[:, 1]
        cxs = u[:, 2] * nx
        cys = u[:, 3] * ny
        q1 = torch.ones(ny, nx, dtype=torch.float64, device=device)
        q2 = torch.empty_like(q1)
        q3 = torch.empty_like(q1)
        i = torch.arange(nx, dtype=torch.float64, device=device)
        for j0 in range(0, ny, rows_per_chunk):
            j1 = min(ny, j0 + rows_per_chunk)
            j = torch.arange(j0, j1, dtype=torch.float64, device=device)
            acc = torch.zeros(j1 - j0, nx, dtype=torch.float64, device=device)
            for g in range(n_gauss):
                ddx = torch.abs(i - cxs[g]); ddx = torch.minimum(ddx, nx - ddx)
                ddy = torch.abs(j - cys[g]); ddy = torch.minimum(ddy, ny - ddy)
                r2 = ddy[:, None] ** 2 + ddx[None, :] ** 2
                acc += amps[g] * torch.exp(-r2 / (2.0 * sigs[g] ** 2))
            q1[j0:j1] += acc
            base = 4 * n_gauss + 2 * j0 * nx
            cnt = (j1 - j0) * nx
            uu = (2.0 * splitmix64_uniform(seed, base, cnt, device=device, stride=2) - 1.0) * (vel / c0)
            vv = (2.0 * splitmix64_uniform(seed, base + 1, cnt, device=device, stride=2) - 1.0) * (vel / c0)
            q2[j0:j1] = q1[j0:j1] * uu.reshape(j1 - j0, nx)
            q3[j0:j1] = q1[j0:j1] * vv.reshape(j1 - j0, nx)
        return q1, q2, q3
    return init


def c3_random(n=4096, steps=200, nu_w=0.8, seed=1311300403, ny=None, name="C3", **kw) -> Workload:
    """C3: random smooth field + grid-scale velocity noise, periodic."""
    nx, ny = n, (n if ny is None else ny)
    dx = LAMBDA_1MHZ / 32
    return Workload(name, nx, ny, dx, dx, dict(MEDIUM_WATER), [(PERIODIC, None)] * 4, 1, nu_w, steps,
                    _multi_gaussian(nx, ny, seed, c0=MEDIUM_WATER["c0"], **kw), f"seed {seed}", extra=dict(seed=seed))


def c5_sweep(n=16384, steps=100, nu_w=0.9, ny=None) -> Workload:
    """C5: throughput sweep; C3's generator (reading A23) with its own seeds per size."""
    seed = {16384: 1311300405, 2048: 1311300406, 8192: 1311300407}.get(n, 1311300405 + 1000 + n)
    return c3_random(n=n, steps=steps, nu_w=nu_w, seed=seed, ny=ny, name=f"C5-{n}")


def c4_hifu(nx=8192, ny=2048, steps=4000, focus_cells=2048.0, aperture_cells=640.0, tau0=None, nu_w=0.8,
            shape=PACKET) -> Workload:
    """C4: focused arc source on x-lo (43a-d) in water, 1 MHz, 1 MPa, extrapolation elsewhere."""
    med = dict(MEDIUM_WATER)
    dx = LAMBDA_1MHZ / 32
    F = focus_cells * dx
    a = aperture_cells * dx
    if tau0 is None:                        # packet numerically zero on the whole aperture at t = 0
        tau0 = -(6.0 + a * a / (2.0 * F * LAMBDA_1MHZ))
    amp = 1.0e6 / (med["rho0"] * med["c0"] ** 2)
    src = _src(shape, amp=amp, freq_hz=1.0e6, focus_m=F, centre_m=ny * dx / 2.0, half_aperture_m=a,
               t0_s=tau0 / 1.0e6)
    return Workload("C4", nx, ny, dx, dx, med, [(SOURCE, src), (EXTRAP, None), (EXTRAP, None), (EXTRAP, None)],
                    1, nu_w, steps, _equilibrium(nx, ny), "HIFU-like packet",
                    extra=dict(tau0=tau0, focus_cells=focus_cells, aperture_cells=aperture_cells))


BY_NAME = {
    "C1": c1_piston,
    "C2": c2_pulse,
    "C3": c3_random,
    "C4": c4_hifu,
    "C5": c5_sweep,
}
