// fvnl_bc.cuh -- ghost-cell rules evaluated on load (no ghost storage), sm_100a.
//
// PAPER.md:326-333 (Dirichlet cells from the analytic profile (41)), PAPER.md:407-420 (focused source (43a-d),
// zero-order extrapolation "simplified absorbing" edges, reflecting border), plus the periodic rule of
// BASELINE.json's configs.  Readings A9, A11, A13, A14, A16 of DESIGN.md.
#pragma once
#include "fvnl_math.cuh"

namespace fvnl {

enum { BC_EXTRAP = 0, BC_PERIODIC = 1, BC_REFLECT = 2, BC_SOURCE = 3 };
enum { SRC_SINE = 0, SRC_PACKET = 1, SRC_TANH = 2 };
enum { SIDE_XLO = 0, SIDE_XHI = 1, SIDE_YLO = 2, SIDE_YHI = 3 };

struct Side {
    int kind, shape;
    double amp, freq_hz, focus_m, centre_m, half_aperture_m, t0_s, steep;
};

// Everything a kernel needs to know about the problem; passed by value (kernel parameter space).
struct Grid {
    int nx, ny;
    double dx, dy, c0, beta, delta;
    Side side[4];
    const double* src;          // analytic ghost cells of this step, written by k_sources (null: no SOURCE side)
};

// Layout of Grid::src (doubles): three ghost layers per SOURCE side, layer l = distance - 1 from the edge; a record is
// (q1, q2, q3), q1 <= 0 marking "outside the aperture" (the cell then behaves as EXTRAP).
//   x-lo, x-hi : record (l, r), rows r = -3 .. ny+2   at  src_off(side) + 3 ((ny + 6) l + r + 3)
//   y-lo, y-hi : record (l, i), columns i = 0 .. nx-1 at  src_off(side) + 3 (nx l + i)
__host__ __device__ inline size_t src_side_doubles(int nx, int ny, int side) { return 9 * (size_t)(side < 2 ? ny + 6 : nx); }
__host__ __device__ inline size_t src_off(int nx, int ny, int side) {
    size_t o = 0;
    for (int s = 0; s < side; ++s) o += src_side_doubles(nx, ny, s);
    return o;
}

// Device-resident clock: the time step lives here so that no host synchronisation is needed between steps
// (dt_n from the CFL number of step n-1).
struct Clock {
    double t;                   // time at the start of the step being computed [s]
    double dt;                  // its time step [s]
    double lamx, lamy;          // c0 dt/dx, c0 dt/dy      (the paper's dt/dx in the units of (20))
    double kapx, kapy;          // delta dt/dx^2, delta dt/dy^2
    double Mprev;               // max |s|/h of the previous step [1/m]; <= 0: unknown
    double last_dt, last_cfl;
    unsigned long long sx_bits, sy_bits;   // running max of |s| in x / y interfaces of the current step (bit patterns)
    long long steps;
    int flags;
    int pad;
};

struct Q3 {
    double q1, q2, q3;
};

// Analytic boundary cell.  side: the edge the ghost cell belongs to; along: coordinate of its centre along that
// edge from the low corner [m]; xc: x of its own centre from the x-lo edge [m] (TANH only).  Returns false when
// the cell is outside the aperture (it then behaves as EXTRAP).
__device__ __noinline__ bool source_cell(const Side& s, int side, double c0, double along, double xc, double t, Q3& out) {
    if (s.shape == SRC_TANH) {                                            // (41), reading A11
        const double q1 = 1.0 - s.amp * tanh(s.steep * (xc - c0 * (t + s.t0_s)));
        out.q1 = q1; out.q2 = q1 - 1.0; out.q3 = 0.0;
        return true;
    }
    const double d = along - s.centre_m;                                   // x2 of (43)
    if (s.half_aperture_m > 0.0 && fabs(d) > s.half_aperture_m) return false;
    const bool focused = (s.focus_m > 0.0) && isfinite(s.focus_m);
    double tau = s.freq_hz * (t + s.t0_s);                                 // periods
    double cth = 1.0, sth = 0.0;
    if (focused) {
        const double lambda_w = c0 / s.freq_hz;
        tau += d * d / (2.0 * s.focus_m * lambda_w);                       // tau = t + x2^2/(2F)
        const double R = sqrt(d * d + s.focus_m * s.focus_m);
        cth = s.focus_m / R;                                               // (43b)
        sth = d / R;                                                       // (43c)
    }
    double g;
    if (s.shape == SRC_SINE) {
        g = (tau >= 0.0) ? s.amp * sin(2.0 * 3.14159265358979323846 * tau) : 0.0;
    } else {                                                               // (43d) with reading A13
        const double e = tau / 4.0;
        const double e2 = e * e, e4 = e2 * e2, e8 = e4 * e4;
        g = s.amp * sin(2.0 * 3.14159265358979323846 * tau) * exp(-(e8 * e2));
    }
    const double qn = g * cth, qt = -g * sth;
    out.q1 = 1.0 + g;                                                      // (43a)
    switch (side) {
        case SIDE_XLO: out.q2 = qn;  out.q3 = qt; break;
        case SIDE_XHI: out.q2 = -qn; out.q3 = qt; break;
        case SIDE_YLO: out.q3 = qn;  out.q2 = qt; break;
        default:       out.q3 = -qn; out.q2 = qt; break;
    }
    return true;
}

__device__ __forceinline__ int wrap(int i, int n) {
    i %= n;
    return i < 0 ? i + n : i;
}
__device__ __forceinline__ int clampi(int i, int n) { return i < 0 ? 0 : (i >= n ? n - 1 : i); }

// Value of the ghost-extended mesh at column i, row r (any integers; the rules are exact for the two ghost
// layers the scheme uses and merely safe beyond them).  The x rule is applied on the y-extended rows, i.e. a
// corner cell is the x-ghost of a y-ghost row (reading A9).  `t` = t_n.
__device__ __forceinline__ Q3 load_ext(const Grid& g, const double* __restrict__ q1, const double* __restrict__ q2,
                                       const double* __restrict__ q3, int i, int r, double t) {
    bool neg2 = false, neg3 = false;
    if (i < 0 || i >= g.nx) {
        const int sd = i < 0 ? SIDE_XLO : SIDE_XHI;
        const int kind = g.side[sd].kind;
        if (kind == BC_PERIODIC) {
            i = wrap(i, g.nx);
        } else if (kind == BC_REFLECT) {
            i = clampi(i < 0 ? -1 - i : 2 * g.nx - 1 - i, g.nx);
            neg2 = true;
        } else {
            if (kind == BC_SOURCE) {
                Q3 c;
                if (source_cell(g.side[sd], sd, g.c0, (r + 0.5) * g.dy, (i + 0.5) * g.dx, t, c)) return c;
            }
            i = clampi(i, g.nx);
        }
    }
    if (r < 0 || r >= g.ny) {
        const int sd = r < 0 ? SIDE_YLO : SIDE_YHI;
        const int kind = g.side[sd].kind;
        if (kind == BC_PERIODIC) {
            r = wrap(r, g.ny);
        } else if (kind == BC_REFLECT) {
            r = clampi(r < 0 ? -1 - r : 2 * g.ny - 1 - r, g.ny);
            neg3 = true;
        } else {
            if (kind == BC_SOURCE) {
                Q3 c;
                if (source_cell(g.side[sd], sd, g.c0, (i + 0.5) * g.dx, (i + 0.5) * g.dx, t, c)) {
                    if (neg2) c.q2 = -c.q2;
                    return c;
                }
            }
            r = clampi(r, g.ny);
        }
    }
    const size_t idx = (size_t)r * g.nx + i;
    Q3 c;
    c.q1 = q1[idx];
    c.q2 = q2[idx];
    c.q3 = q3[idx];
    if (neg2) c.q2 = -c.q2;
    if (neg3) c.q3 = -c.q3;
    return c;
}

// One-deep ghost of an intermediate state for the source step (26) (reading A9): the rule of `sd` applied to the
// interior value `inner` (the cell next to the edge, or the wrapped one for PERIODIC -- the caller passes it).
// `along`, `xc`: as for source_cell.
__device__ __forceinline__ Q3 ghost_of(const Grid& g, int sd, const Q3& inner, double along, double xc, double t) {
    const int kind = g.side[sd].kind;
    Q3 c = inner;
    if (kind == BC_REFLECT) {
        if (sd < 2) c.q2 = -c.q2; else c.q3 = -c.q3;
    } else if (kind == BC_SOURCE) {
        Q3 s;
        if (source_cell(g.side[sd], sd, g.c0, along, xc, t, s)) c = s;
    }
    return c;
}

}  // namespace fvnl
