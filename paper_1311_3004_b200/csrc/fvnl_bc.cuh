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
    double amp, freq_hz, focus_m, centre_m, half_aperture_m, t0_s, steep, theta;
};

// Everything a kernel needs to know about the problem; passed by value (kernel parameter space).
struct Grid {
    int nx, ny;
    double dx, dy, c0, beta, delta;
    double x0;                  // x of the x-lo edge in the frame of the travelling profile (41); moves with fvnl_shift
    Side side[4];
    double* src;                // analytic ghost cells of SOURCE sides: two buffers (below), null without a SOURCE side
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
// Two such buffers, used alternately: step n reads buffer n & 1 (values at t_n) while its blocks already write buffer
// (n + 1) & 1 with the values at t_{n+1} = t_n + dt_n, which is known when step n starts (dt is lagged).
__host__ __device__ inline size_t src_stride(int nx, int ny) { return (src_off(nx, ny, 4) + 31) / 32 * 32; }
__host__ __device__ inline double* src_buffer(const Grid& g, long long step) {
    return g.src ? g.src + (size_t)(step & 1) * src_stride(g.nx, g.ny) : nullptr;
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
    unsigned int ticket;        // blocks of the running step kernel that have finished (the last one ends the step)
};

// dt of the step about to start and everything derived from it.  mode 0: value = dt; mode 1: value = nu_W and
// dt = nu_W / (c0 M), M = max |s|/h of the previous step (reading A7).  Also clears the running maxima.
__device__ __forceinline__ void clock_set_dt(const Grid& g, Clock* c, double value, int mode, double M) {
    const double dt = (mode == 1) ? __ddiv_rn(value, __dmul_rn(g.c0, M)) : value;
    c->dt = dt;
    c->lamx = __ddiv_rn(__dmul_rn(g.c0, dt), g.dx);
    c->lamy = __ddiv_rn(__dmul_rn(g.c0, dt), g.dy);
    c->kapx = __ddiv_rn(__dmul_rn(g.delta, dt), __dmul_rn(g.dx, g.dx));
    c->kapy = __ddiv_rn(__dmul_rn(g.delta, dt), __dmul_rn(g.dy, g.dy));
    if (__dadd_rn(c->kapx, c->kapy) > 0.5) c->flags |= F_ECFL;
    if (!(dt > 0.0) || not_finite(dt)) c->flags |= F_ENAN;
    c->sx_bits = 0ull;
    c->sy_bits = 0ull;
    c->ticket = 0u;
}

// End of step n: M_n from the running maxima, nu_n, t_{n+1}; and, when another step of the same call follows, its dt.
__device__ __forceinline__ void clock_advance(const Grid& g, Clock* c, double value, int mode, int more) {
    const double sx = __longlong_as_double((long long)*(volatile unsigned long long*)&c->sx_bits);
    const double sy = __longlong_as_double((long long)*(volatile unsigned long long*)&c->sy_bits);
    const double M = fmax(__ddiv_rn(sx, g.dx), __ddiv_rn(sy, g.dy));
    c->last_dt = c->dt;
    c->last_cfl = __dmul_rn(__dmul_rn(g.c0, c->dt), M);
    if (c->last_cfl > 1.0) c->flags |= F_ECFL;
    c->Mprev = M;
    c->t = __dadd_rn(c->t, c->dt);
    c->steps += 1;
    c->ticket = 0u;
    if (more) clock_set_dt(g, c, value, mode, M);
}

struct Q3 {
    double q1, q2, q3;
};

// Analytic boundary cell: the value an edge of kind SOURCE prescribes for one of its ghost cells at time t.
//   side   the edge the ghost cell belongs to;
//   along  coordinate of the cell's centre along that edge, from the low corner [m];
//   xc, yc the cell's own centre [m]: x in the frame of the profile (41) (Grid::x0 + distance from the x-lo edge), y from the
//          y-lo edge (used by the travelling profile only).
// Returns false for a cell outside the aperture: it then follows the extrapolation rule.
//
// (41), PAPER.md:330 (reading A11): the travelling profile rho' = -K tanh(k (xi - c0 t')) moving along the unit vector
// e = (cos theta_T, sin theta_T), xi = (x, y).e ("a standard rotation change of variables"), with the
// velocity along e: (q2, q3) = rho' e  (theta_T = 0: q2 = q1 - 1, q3 = 0 as printed).
//
// (43a-d), written from the geometry the paper describes rather than from its component formulas:
// the transducer is a circular arc centred on the focus; the focus lies at distance F from the edge on the inward normal
// through the centre of the aperture.  Seen from the edge point at signed distance x2 from that centre, the focus is in
// the direction  F n - x2 e  (n: inward normal, e: along the edge), at distance hypot(F, x2).  The arc emits towards the
// focus, so the momentum is g times the unit vector of that direction and the density is 1 + g; the point fires ahead of
// the centre by the extra path, in the paraxial form the paper gives:  phase = f t' + x2^2 / (2 F lambda)  [periods].
// g = A sin(2 pi phase) (piston, switched on at phase 0) or the same carrier under the packet envelope exp(-(phase/4)^10)
// (reading A13).  F <= 0 or infinite: plane wave, direction n, no phase lead.
__device__ __noinline__ bool source_cell(const Side& s, int side, double c0, double along, double xc, double yc, double t,
                                         Q3& out) {
    const double tp = t + s.t0_s;
    if (s.shape == SRC_TANH) {
        double e_y, e_x;
        sincos(s.theta, &e_y, &e_x);
        const double xi = fma(xc, e_x, yc * e_y);
        out.q1 = 1.0 - s.amp * tanh(s.steep * fma(-c0, tp, xi));
        const double rho1 = out.q1 - 1.0;                                             // of the ROUNDED q1, as (41) has it
        out.q2 = rho1 * e_x; out.q3 = rho1 * e_y + 0.0;
        return true;
    }
    const double x2 = along - s.centre_m;
    if (s.half_aperture_m > 0.0 && fabs(x2) > s.half_aperture_m) return false;
    double phase = s.freq_hz * tp;
    double to_focus_n = 1.0, to_focus_e = 0.0;                                        // unit vector towards the focus
    if (s.focus_m > 0.0 && s.focus_m <= 1.7976931348623157e308) {
        const double inv_dist = rhypot(s.focus_m, x2);
        to_focus_n = s.focus_m * inv_dist;
        to_focus_e = -x2 * inv_dist;
        phase += (x2 / s.focus_m) * (x2 * s.freq_hz / c0) * 0.5;                      // x2^2/(2 F lambda), lambda = c0/f
    }
    double g = s.amp * sinpi(2.0 * phase);
    if (s.shape == SRC_PACKET) {
        const double w = 0.25 * phase, w2 = w * w, w5 = w2 * w2 * w;
        g *= exp(-(w5 * w5));
    } else if (phase < 0.0) {
        g = 0.0;
    }
    const double m_n = (side & 1) ? -g * to_focus_n : g * to_focus_n;                 // hi sides: the inward normal is -x / -y
    const double m_e = g * to_focus_e;
    out.q1 = 1.0 + g;
    if (side < 2) { out.q2 = m_n; out.q3 = m_e; }                                     // x sides: normal = x
    else          { out.q2 = m_e; out.q3 = m_n; }                                     // y sides: normal = y
    return true;
}

// The analytic cell of SOURCE side sd at position (column i, row r) of the ghost-extended mesh.
__device__ __forceinline__ bool source_at(const Grid& g, int sd, int i, int r, double t, Q3& out) {
    const double x = (i + 0.5) * g.dx, y = (r + 0.5) * g.dy;
    return source_cell(g.side[sd], sd, g.c0, sd < 2 ? y : x, g.x0 + x, y, t, out);
}

// Record n of Grid::src (layout above): the analytic cell of one ghost position at time t; q1 = -1 marks "outside the
// aperture" (and a record of a side that is not a SOURCE).  n < src_off(nx, ny, 4) / 3.
__device__ __forceinline__ Q3 source_record_value(const Grid& g, double t, size_t n) {
    Q3 none;
    none.q1 = -1.0; none.q2 = 0.0; none.q3 = 0.0;
    size_t m = n;
    for (int sd = 0; sd < 4; ++sd) {
        const size_t recs = src_side_doubles(g.nx, g.ny, sd) / 3;
        if (m < recs) {
            if (g.side[sd].kind != BC_SOURCE) return none;
            const int per = sd < 2 ? g.ny + 6 : g.nx;
            const int layer = (int)(m / per), pos = (int)(m % per);
            Q3 c;
            bool in;
            if (sd < 2) in = source_at(g, sd, sd == SIDE_XLO ? -1 - layer : g.nx + layer, pos - 3, t, c);
            else in = source_at(g, sd, pos, sd == SIDE_YLO ? -1 - layer : g.ny + layer, t, c);
            return in ? c : none;
        }
        m -= recs;
    }
    return none;
}
__device__ __forceinline__ void source_record(const Grid& g, double t, size_t n, double* __restrict__ out) {
    for (int sd = 0, m = 0; sd < 4; ++sd) {                    // (records of sides that are not a SOURCE are never read)
        m += (int)(src_side_doubles(g.nx, g.ny, sd) / 3);
        if (n < (size_t)m) { if (g.side[sd].kind != BC_SOURCE) return; break; }
    }
    const Q3 c = source_record_value(g, t, n);
    double* o = out + 3 * n;
    o[0] = c.q1; o[1] = c.q2; o[2] = c.q3;
}
// Index of the record of ghost layer l (0 = next to the edge) of SOURCE side sd at position pos (row for an x side, column
// for a y side).
__host__ __device__ inline size_t src_record_index(int nx, int ny, int sd, int layer, int pos) {
    return src_off(nx, ny, sd) / 3 + (sd < 2 ? (size_t)(ny + 6) * layer + (pos + 3) : (size_t)nx * layer + pos);
}

__device__ __forceinline__ int wrap(int i, int n) {
    i %= n;
    return i < 0 ? i + n : i;
}
__device__ __forceinline__ int clampi(int i, int n) { return i < 0 ? 0 : (i >= n ? n - 1 : i); }

// Value of the ghost-extended mesh at column i, row r (any integers; the rules are exact for the two ghost
// layers the scheme uses and merely safe beyond them).  The x rule is applied on the y-extended rows, i.e. a
// corner cell is the x-ghost of a y-ghost row (reading A9).  `t` = t_n.
// `cells`: where the interior cells live -- any callable idx -> Q3 (idx = row * nx + column).
template <class Cells>
__device__ __forceinline__ Q3 load_ext(const Grid& g, const Cells& cells, int i, int r, double t) {
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
                if (source_at(g, sd, i, r, t, c)) return c;
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
                if (source_at(g, sd, i, r, t, c)) {
                    if (neg2) c.q2 = -c.q2;
                    return c;
                }
            }
            r = clampi(r, g.ny);
        }
    }
    Q3 c = cells((size_t)r * g.nx + i);
    if (neg2) c.q2 = -c.q2;
    if (neg3) c.q3 = -c.q3;
    return c;
}

// Three planes in (global) memory, structure of arrays.
struct PlaneCells {
    const double *q1, *q2, *q3;
    __device__ __forceinline__ Q3 operator()(size_t idx) const {
        Q3 c;
        c.q1 = q1[idx]; c.q2 = q2[idx]; c.q3 = q3[idx];
        return c;
    }
};
struct PlaneOut {
    double *q1, *q2, *q3;
    __device__ __forceinline__ void put(size_t idx, const Q3& c) const { q1[idx] = c.q1; q2[idx] = c.q2; q3[idx] = c.q3; }
};


// One-deep ghost of an intermediate state for the source step (26) (reading A9): the rule of `sd` applied to the
// interior value `inner` (the cell next to the edge, or the wrapped one for PERIODIC -- the caller passes it).
// (i, r): the ghost cell's position on the ghost-extended mesh.
__device__ __forceinline__ Q3 ghost_of(const Grid& g, int sd, const Q3& inner, int i, int r, double t) {
    const int kind = g.side[sd].kind;
    Q3 c = inner;
    if (kind == BC_REFLECT) {
        if (sd < 2) c.q2 = -c.q2; else c.q3 = -c.q3;
    } else if (kind == BC_SOURCE) {
        Q3 s;
        if (source_at(g, sd, i, r, t, s)) c = s;
    }
    return c;
}

}  // namespace fvnl
