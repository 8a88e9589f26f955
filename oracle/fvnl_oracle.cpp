// fvnl_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, serial CPU oracle for the per-time-step 2-D high-resolution
// finite-volume update of arXiv 1311.3004 (Velasco-Segura & Rendon), written
// from the paper (/root/reference/PAPER.md; "PAPER.md:<line>" below) in the
// paper's order and notation.  fp64, one operation per formula, no blocking,
// no fusion, ghost arrays materialised.  It shares no code, header, table or
// constant with the CUDA path under paper_1311_3004_b200/csrc/, and nothing
// under paper_1311_3004_b200/ may import, link or execute it.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// call it.
//
// Build:  g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC   (oracle/build.py)
//   -ffp-contract=off: no FMA contraction, every formula rounds as written.
//   OpenMP only distributes independent rows / columns over threads; each row
//   or column is computed by exactly the serial code, so the state is bitwise
//   identical for any thread count (max is order independent).  orc_set_threads(1)
//   gives the serial oracle.
//
// Pins (tests/test_oracle_pins.py, `-m "not gpu"`): Table I row theta_T = 0
// (PAPER.md:345-354), Roe property (31), conservation
// (PAPER.md:127), mirror symmetry, shear-mode decay, Fubini 2nd harmonic,
// nu = 1 shift, first-order speeds (36)-(38), region S
// (PAPER.md:263-267), numerical eigen-decomposition of the printed Roe matrix
// (PAPER.md:233), the 4x4 worked step (tests/golden/p9_4x4.txt).
// PARITY UNPINNED (no number in the paper fixes them):
// ghost policy between sub-steps under non-periodic BC (A9), the envelope
// exponent of (43d) (A13), where ghost layers sample (43) (A14).
//
// State: dimensionless q of (22): q1 = rho/rho0,
// q2 = q1*u/c0, q3 = q1*v/c0.  Layout: three planes of nx*ny doubles,
// idx = j*nx + i, i = x index (fastest).

#include <cmath>
#include <cstddef>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- status / flag values of the oracle's own interface --------------------
enum { ORC_OK = 0, ORC_EARG = 1, ORC_ECFL = 16, ORC_ENONREAL = 32, ORC_ENONPOS = 64, ORC_ENAN = 128 };
enum { BC_EXTRAP = 0, BC_PERIODIC = 1, BC_REFLECT = 2, BC_SOURCE = 3 };
enum { SRC_SINE = 0, SRC_PACKET = 1, SRC_TANH = 2 };
enum { SIDE_XLO = 0, SIDE_XHI = 1, SIDE_YLO = 2, SIDE_YHI = 3 };

struct Source {
    int shape;
    double amp, freq_hz, focus_m, centre_m, half_aperture_m, t0_s, steep;
    double theta;     // TANH only: propagation angle theta_T from the x_1 axis
};

struct Cell { double q[3]; };

// One interface's Riemann solution.
struct Riemann {
    double s[3];      // speeds s^1, s^2, s^3  (32)-(34)
    double W[3][3];   // waves W^p = alpha^p r^p, W[p][component]
    double amdq[3];   // A^- Delta Q  (28)
    double apdq[3];   // A^+ Delta Q  (29)
    int flag;
};

// ---------------------------------------------------------------------------
// Flux f_1 of (22):  f_j = q^{j+1}/(q^1)^2 (  (q^1)^2, q^2, q^3 ) + phi (0, d1j, d2j),
// phi = q^1 + (beta-1)(q^1-1)^2.   dir = 0: f_1, dir = 1: f_2.
void flux(const double q[3], double beta, int dir, double f[3]) {
    const double q1 = q[0];
    const double qn = q[1 + dir];
    const double phi = q1 + (beta - 1.0) * (q1 - 1.0) * (q1 - 1.0);
    const double c = qn / (q1 * q1);
    f[0] = c * (q1 * q1);
    f[1] = c * q[1];
    f[2] = c * q[2];
    f[1 + dir] += phi;
}

// ---------------------------------------------------------------------------
// Roe-linearised Riemann solve between QL (cell i-1) and QR (cell i), x-direction form.
// PAPER.md:218-245.  Eigenvectors (not printed, "straightforward"):
// solving  A r = s r  for the printed matrix with first component 1 gives
//   r^{1,2} = ( 1, s, (Zb3/Zb1)(s - 2 Zb2)/(s - v) ),  v = Zb2/Zb1,  s - v = +-a ;   r^3 = (0,0,1).
void riemann(const double QL[3], const double QR[3], double beta, Riemann& R) {
    R.flag = 0;
    // primitive variables z = (q1, q2/q1, q3/q1)
    const double zL[3] = { QL[0], QL[1] / QL[0], QL[2] / QL[0] };
    const double zR[3] = { QR[0], QR[1] / QR[0], QR[2] / QR[0] };
    if (!(QL[0] > 0.0) || !(QR[0] > 0.0)) R.flag |= ORC_ENONPOS;
    // arithmetic means Zbar^p = (Z_i^p + Z_{i-1}^p)/2 ,  Phi = 1 + 2(beta-1)(Zbar^1 - 1)
    const double Zb1 = 0.5 * (zR[0] + zL[0]);
    const double Zb2 = 0.5 * (zR[1] + zL[1]);
    const double Zb3 = 0.5 * (zR[2] + zL[2]);
    const double Phi = 1.0 + 2.0 * (beta - 1.0) * (Zb1 - 1.0);
    // eigenvalues (32)-(34)
    const double v = Zb2 / Zb1;
    const double disc = (Zb2 * Zb2) / (Zb1 * Zb1) - 2.0 * (Zb2 * Zb2) / Zb1 + Phi;
    if (disc < 0.0) R.flag |= ORC_ENONREAL;
    const double a = std::sqrt(disc);
    const double s1 = v + a, s2 = v - a, s3 = v;
    R.s[0] = s1; R.s[1] = s2; R.s[2] = s3;
    // third components of r^1, r^2
    const double w = Zb3 / Zb1;
    const double r31 = w * (s1 - 2.0 * Zb2) / a;      // (s1 - v) = +a
    const double r32 = -w * (s2 - 2.0 * Zb2) / a;     // (s2 - v) = -a
    // Q_i - Q_{i-1} = sum_p alpha^p r^p
    const double D1 = QR[0] - QL[0], D2 = QR[1] - QL[1], D3 = QR[2] - QL[2];
    const double al1 = (D2 - s2 * D1) / (2.0 * a);
    const double al2 = (s1 * D1 - D2) / (2.0 * a);
    const double al3 = D3 - al1 * r31 - al2 * r32;
    // waves W^p = alpha^p r^p
    R.W[0][0] = al1;  R.W[0][1] = al1 * s1;  R.W[0][2] = al1 * r31;
    R.W[1][0] = al2;  R.W[1][1] = al2 * s2;  R.W[1][2] = al2 * r32;
    R.W[2][0] = 0.0;  R.W[2][1] = 0.0;       R.W[2][2] = al3;
    // fluctuations (28), (29)
    for (int m = 0; m < 3; ++m) { R.amdq[m] = 0.0; R.apdq[m] = 0.0; }
    for (int p = 0; p < 3; ++p) {
        const double sm = std::min(R.s[p], 0.0), sp = std::max(R.s[p], 0.0);
        for (int m = 0; m < 3; ++m) {
            R.amdq[m] += sm * R.W[p][m];
            R.apdq[m] += sp * R.W[p][m];
        }
    }
    if (!(disc == disc)) R.flag |= ORC_ENAN;
}

// monotonized central-difference limiter
double mc_phi(double theta) {
    return std::max(0.0, std::min(std::min((1.0 + theta) / 2.0, 2.0), 2.0 * theta));
}

// ---------------------------------------------------------------------------
// SWEEP: one row (or column) of (27) with (28)-(30).  PAPER.md:159-198.
// cells[0..n+3] = 2 ghosts | n interior | 2 ghosts (already in x-form: for the y-sweep the caller
// has switched positions 2 and 3).  lam = Delta t / Delta x in the paper's units.
// out[0..n-1] = updated interior.  smax = max over interfaces touching >= 1 interior cell of
// max(|s^1|,|s^2|,|s^3|).
void sweep(int n, const Cell* cells, double lam, double beta, Cell* out, double* smax, int* flag) {
    const int nif = n + 3;                 // interfaces k = 0..n+2 ; interface k lies between cells[k], cells[k+1]
    std::vector<Riemann> R(nif);
    for (int k = 0; k < nif; ++k) {
        riemann(cells[k].q, cells[k + 1].q, beta, R[k]);
        *flag |= R[k].flag;
    }
    // correction fluxes (30) at the n+1 interfaces that touch an interior cell: k = 1..n+1
    std::vector<Cell> Ft(nif);
    for (int k = 1; k <= n + 1; ++k) {
        double F[3] = { 0.0, 0.0, 0.0 };
        for (int p = 0; p < 3; ++p) {
            const double* Wk = R[k].W[p];
            const double nrm = Wk[0] * Wk[0] + Wk[1] * Wk[1] + Wk[2] * Wk[2];
            double phi = 0.0;
            if (nrm != 0.0) {
                const int K = (R[k].s[p] > 0.0) ? k - 1 : k + 1;        // upwind interface I
                const double* WK = R[K].W[p];
                const double theta = (WK[0] * Wk[0] + WK[1] * Wk[1] + WK[2] * Wk[2]) / nrm;
                phi = mc_phi(theta);
            }
            const double as = std::fabs(R[k].s[p]);
            const double c = 0.5 * as * (1.0 - lam * as);               // (30)
            for (int m = 0; m < 3; ++m) F[m] += c * phi * Wk[m];
        }
        for (int m = 0; m < 3; ++m) Ft[k].q[m] = F[m];
        const double sm = std::max(std::fabs(R[k].s[0]), std::max(std::fabs(R[k].s[1]), std::fabs(R[k].s[2])));
        if (sm > *smax) *smax = sm;
        if (!(sm == sm)) *flag |= ORC_ENAN;
    }
    // update (27)   PAPER.md:161 : interior cell c (0-based) = cells[c+2]; its left interface is k = c+1, right k = c+2
    for (int c = 0; c < n; ++c) {
        const int kl = c + 1, kr = c + 2;
        for (int m = 0; m < 3; ++m) {
            out[c].q[m] = cells[c + 2].q[m]
                        - lam * (R[kr].amdq[m] + R[kl].apdq[m])
                        - lam * (Ft[kr].q[m] - Ft[kl].q[m]);
        }
    }
}

// ---------------------------------------------------------------------------
struct Oracle {
    int nx, ny;
    double dx, dy;
    double c0, rho0, beta, delta;
    int bc[4];
    Source src[4];
    std::vector<double> q[3];
    double t, M_prev, last_dt, last_cfl;
    double x_origin;  // x of the x-lo edge in the frame in which the travelling profile (41) is written; moves with the
                      // domain in the second stage
    long steps;
    int flags;
    int nthreads;
};

inline Cell load(const std::vector<double>* q, size_t idx) {
    Cell c; c.q[0] = q[0][idx]; c.q[1] = q[1][idx]; c.q[2] = q[2][idx]; return c;
}

// Boundary source cell.  (41) PAPER.md:330 ; (43a-d) PAPER.md:409-418 ; readings A11, A13, A14, A16.
// side: which edge the ghost cell belongs to.  along_m: coordinate of the cell centre along that edge, measured
// from the low corner.  xc_m, yc_m: x and y of the ghost cell's own centre measured from the x-lo / y-lo edge (TANH only).
// Returns false if the cell lies outside the aperture (then it behaves as EXTRAP).
bool source_cell(const Oracle& o, int side, double along_m, double xc_m, double yc_m, double t, Cell* out) {
    const Source& s = o.src[side];
    const double PI = 3.14159265358979323846;
    if (s.shape == SRC_TANH) {
        // q1 = 1 - (delta~/beta) tanh(x - t), q2 = q1 - 1, q3 = 0 in the paper's units (41); "steep" carries the 10%-90%
        // width (A11).  Propagation at an angle theta_T from the x_1 axis: "to use them with a different value of theta_T,
        // we have applied a standard rotation change of variables": x -> the coordinate along the
        // propagation direction, x cos(theta) + y sin(theta); the velocity (q2, q3) -> its rotation by theta.
        const double ct = std::cos(s.theta), st = std::sin(s.theta);
        const double xi = (o.x_origin + xc_m) * ct + yc_m * st;
        const double q1 = 1.0 - s.amp * std::tanh(s.steep * (xi - o.c0 * (t + s.t0_s)));
        out->q[0] = q1; out->q[1] = (q1 - 1.0) * ct; out->q[2] = (q1 - 1.0) * st + 0.0;
        return true;
    }
    const double d = along_m - s.centre_m;                       // x_2 of (43), from the aperture centre
    if (s.half_aperture_m > 0.0 && std::fabs(d) > s.half_aperture_m) return false;
    const bool focused = (s.focus_m > 0.0) && std::isfinite(s.focus_m);
    const double lambda_w = o.c0 / s.freq_hz;
    double tau = s.freq_hz * (t + s.t0_s);                       // time in periods
    double cth = 1.0, sth = 0.0;
    if (focused) {
        tau += d * d / (2.0 * s.focus_m * lambda_w);             // tau = t + x_2^2/(2F)
        const double R = std::sqrt(d * d + s.focus_m * s.focus_m);
        cth = s.focus_m / R;                                     // F/sqrt(x_2^2+F^2)     (43b)
        sth = d / R;                                             // x_2/sqrt(x_2^2+F^2)   (43c)
    }
    double g;
    if (s.shape == SRC_SINE) {
        g = (tau >= 0.0) ? s.amp * std::sin(2.0 * PI * tau) : 0.0;
    } else {                                                     // SRC_PACKET (43d) with A13: exp(-(tau/4)^10)
        const double e = tau / 4.0;
        const double e2 = e * e, e4 = e2 * e2, e8 = e4 * e4;
        g = s.amp * std::sin(2.0 * PI * tau) * std::exp(-(e8 * e2));
    }
    const double qn = g * cth;                                   // momentum along the inward normal
    const double qt = -g * sth;                                  // momentum along the edge (towards the centre)
    out->q[0] = 1.0 + g;                                         // (43a)
    switch (side) {
        case SIDE_XLO: out->q[1] =  qn; out->q[2] = qt; break;
        case SIDE_XHI: out->q[1] = -qn; out->q[2] = qt; break;
        case SIDE_YLO: out->q[2] =  qn; out->q[1] = qt; break;
        default:       out->q[2] = -qn; out->q[1] = qt; break;
    }
    return true;
}

// Ghost rule G(.) for one line of cells along `axis` (0: a row j = fixed, 1: a column i = fixed).
// line[0..n-1] interior values (already gathered), depth g ghosts each side written to lo[0..g-1] (lo[0] nearest
// the interior ... lo[g-1] outermost) and hi[0..g-1] likewise.   `fixed` = index of the row / column.
// PAPER.md:326-333 (Dirichlet from (41)), 407-420 (source + zero-order extrapolation + reflecting border).
void ghosts(const Oracle& o, int axis, int fixed, const Cell* line, int n, int g, double t, Cell* lo, Cell* hi) {
    const int side_lo = (axis == 0) ? SIDE_XLO : SIDE_YLO;
    const int side_hi = side_lo + 1;
    const int ncomp = 1 + axis;                                   // momentum component normal to these edges
    const double h_along = (axis == 0) ? o.dy : o.dx;             // spacing along the edge
    for (int e = 0; e < 2; ++e) {
        const int side = e ? side_hi : side_lo;
        Cell* G = e ? hi : lo;
        for (int k = 0; k < g; ++k) {
            Cell c;
            const int kind = o.bc[side];
            if (kind == BC_PERIODIC) {
                c = e ? line[k] : line[n - 1 - k];
            } else if (kind == BC_REFLECT) {
                c = e ? line[n - 1 - k] : line[k];
                c.q[ncomp] = -c.q[ncomp];
            } else {
                c = e ? line[n - 1] : line[0];                    // zero-order extrapolation
                if (kind == BC_SOURCE) {
                    const double along = (fixed + 0.5) * h_along;
                    // x, y of this ghost cell's own centre from the x-lo / y-lo edge (TANH)
                    double xc, yc;
                    if (axis == 0) { xc = e ? (o.nx + k + 0.5) * o.dx : -(k + 0.5) * o.dx; yc = (fixed + 0.5) * o.dy; }
                    else           { xc = (fixed + 0.5) * o.dx; yc = e ? (o.ny + k + 0.5) * o.dy : -(k + 0.5) * o.dy; }
                    Cell sc;
                    if (source_cell(o, side, along, xc, yc, t, &sc)) c = sc;
                }
            }
            G[k] = c;
        }
    }
}

inline void swap23(Cell& c) { std::swap(c.q[1], c.q[2]); }

// Gather one line of the mesh (axis 0: row `l`, axis 1: column `l`) into cells[2..n+1] and fill the 2+2 ghosts.
void gather_line(const Oracle& o, int axis, int l, std::vector<Cell>& cells) {
    const int n = axis == 0 ? o.nx : o.ny;
    cells.resize(n + 4);
    for (int c = 0; c < n; ++c) {
        const size_t idx = axis == 0 ? (size_t)l * o.nx + c : (size_t)c * o.nx + l;
        cells[c + 2] = load(o.q, idx);
    }
    Cell lo[2], hi[2];
    ghosts(o, axis, l, &cells[2], n, 2, o.t, lo, hi);
    cells[1] = lo[0]; cells[0] = lo[1]; cells[n + 2] = hi[0]; cells[n + 3] = hi[1];
}

// O2: x-sweep (24) over the y-extended mesh, and O3: y-sweep (25) with positions 2 and 3 switched
// (PAPER.md:155, 271).  Reading A9: the ghost cells are filled from Q^n, sources at t_n, and --
// following the CLAWPACK logic the paper says it follows -- the x-sweep also runs over the two
// ghost rows beyond each y edge, so that the ghost rows the y-sweep sees are at the same intermediate level Q*
// as the interior.  For EXTRAP / PERIODIC / REFLECT edges this is identical to applying the ghost rule to Q*;
// for an analytic edge (41) it is what keeps the y-ghost rows in step with the interior (Table I, PAPER.md:345-354,
// is not reproducible otherwise).
// Returns M = max |s|/h over the interfaces that touch an interior cell, both directions (A8).
double sweeps(Oracle& o, double dt, int stages) {
    const int nx = o.nx, ny = o.ny;
    const double lamx = o.c0 * dt / o.dx;                         // Delta t/Delta x in the units of (20)
    const double lamy = o.c0 * dt / o.dy;
    double sx_all = 0.0, sy_all = 0.0;
    int flag_all = 0;

    // y-extended copy of Q^n: rows -2..ny+1 (row r stored at r+2), ghost rows by the y-side rule at t_n
    std::vector<Cell> ext((size_t)(ny + 4) * nx);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) ext[(size_t)(j + 2) * nx + i] = load(o.q, (size_t)j * nx + i);
    for (int i = 0; i < nx; ++i) {
        std::vector<Cell> col(ny);
        for (int j = 0; j < ny; ++j) col[j] = ext[(size_t)(j + 2) * nx + i];
        Cell lo[2], hi[2];
        ghosts(o, 1, i, col.data(), ny, 2, o.t, lo, hi);
        ext[(size_t)1 * nx + i] = lo[0]; ext[(size_t)0 * nx + i] = lo[1];
        ext[(size_t)(ny + 2) * nx + i] = hi[0]; ext[(size_t)(ny + 3) * nx + i] = hi[1];
    }

    // O2: Q* = x-sweep of every row of the extended mesh
    std::vector<Cell> star((size_t)(ny + 4) * nx);
    if (stages & 1) {
#pragma omp parallel for schedule(static) reduction(max : sx_all) reduction(| : flag_all) num_threads(o.nthreads)
        for (int r = -2; r < ny + 2; ++r) {
            std::vector<Cell> cells(nx + 4), res(nx);
            for (int i = 0; i < nx; ++i) cells[i + 2] = ext[(size_t)(r + 2) * nx + i];
            Cell lo[2], hi[2];
            ghosts(o, 0, r, &cells[2], nx, 2, o.t, lo, hi);
            cells[1] = lo[0]; cells[0] = lo[1]; cells[nx + 2] = hi[0]; cells[nx + 3] = hi[1];
            double smax = 0.0; int flag = 0;
            sweep(nx, cells.data(), lamx, o.beta, res.data(), &smax, &flag);
            for (int i = 0; i < nx; ++i) star[(size_t)(r + 2) * nx + i] = res[i];
            if (r >= 0 && r < ny) {                               // ghost rows do not enter M
                if (smax > sx_all) sx_all = smax;
                flag_all |= flag;
            }
        }
    } else {
        star = ext;
    }

    // O3: Q** = y-sweep of every column of Q* (components 2 and 3 switched on entry and exit)
    if (stages & 2) {
        std::vector<double> out[3];
        for (int m = 0; m < 3; ++m) out[m].resize(o.q[m].size());
#pragma omp parallel for schedule(static) reduction(max : sy_all) reduction(| : flag_all) num_threads(o.nthreads)
        for (int i = 0; i < nx; ++i) {
            std::vector<Cell> cells(ny + 4), res(ny);
            for (int r = 0; r < ny + 4; ++r) { cells[r] = star[(size_t)r * nx + i]; swap23(cells[r]); }
            double smax = 0.0; int flag = 0;
            sweep(ny, cells.data(), lamy, o.beta, res.data(), &smax, &flag);
            for (int j = 0; j < ny; ++j) {
                swap23(res[j]);
                for (int m = 0; m < 3; ++m) out[m][(size_t)j * nx + i] = res[j].q[m];
            }
            if (smax > sy_all) sy_all = smax;
            flag_all |= flag;
        }
        for (int m = 0; m < 3; ++m) o.q[m].swap(out[m]);
    } else {
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                for (int m = 0; m < 3; ++m) o.q[m][(size_t)j * nx + i] = star[(size_t)(j + 2) * nx + i].q[m];
    }
    o.flags |= flag_all;
    return std::max(sx_all / o.dx, sy_all / o.dy);
}

// O7: pre-pass.  M of the current state, x-interfaces of G_x(Q) and y-interfaces of G_y(Q), no update.
double prepass(Oracle& o) {
    double m_all = 0.0;
    int flag_all = 0;
    for (int axis = 0; axis < 2; ++axis) {
        const int nl = axis == 0 ? o.ny : o.nx;
        const int n = axis == 0 ? o.nx : o.ny;
        const double h = axis == 0 ? o.dx : o.dy;
#pragma omp parallel for schedule(static) reduction(max : m_all) reduction(| : flag_all) num_threads(o.nthreads)
        for (int l = 0; l < nl; ++l) {
            std::vector<Cell> cells, res(n);
            gather_line(o, axis, l, cells);
            if (axis == 1) for (auto& c : cells) swap23(c);
            double smax = 0.0; int flag = 0;
            sweep(n, cells.data(), 0.0, o.beta, res.data(), &smax, &flag);
            if (smax / h > m_all) m_all = smax / h;
            flag_all |= flag;
        }
    }
    o.flags |= flag_all;
    return m_all;
}

// O4: source step (26), psi = delta~ (0, lap(q2/q1), lap(q3/q1)) (reading A1), "standard central
// finite difference second-order": 5-point Laplacian, one forward-Euler step (reading A2).
void source_step(Oracle& o, double dt) {
    const int nx = o.nx, ny = o.ny;
    const double kx = o.delta * dt / (o.dx * o.dx);
    const double ky = o.delta * dt / (o.dy * o.dy);
    // ghost-extended primitive fields z^2, z^3 of the current (intermediate) state, 1 ghost deep; corners unused
    const int sx = nx + 2;
    std::vector<double> z2((size_t)sx * (ny + 2), 0.0), z3((size_t)sx * (ny + 2), 0.0);
    auto Z = [&](std::vector<double>& z, int i, int j) -> double& { return z[(size_t)(j + 1) * sx + (i + 1)]; };
#pragma omp parallel for schedule(static) num_threads(o.nthreads)
    for (int j = 0; j < ny; ++j) {
        std::vector<Cell> row(nx);
        for (int i = 0; i < nx; ++i) row[i] = load(o.q, (size_t)j * nx + i);
        Cell lo[1], hi[1];
        ghosts(o, 0, j, row.data(), nx, 1, o.t, lo, hi);
        for (int i = 0; i < nx; ++i) { Z(z2, i, j) = row[i].q[1] / row[i].q[0]; Z(z3, i, j) = row[i].q[2] / row[i].q[0]; }
        Z(z2, -1, j) = lo[0].q[1] / lo[0].q[0]; Z(z3, -1, j) = lo[0].q[2] / lo[0].q[0];
        Z(z2, nx, j) = hi[0].q[1] / hi[0].q[0]; Z(z3, nx, j) = hi[0].q[2] / hi[0].q[0];
    }
#pragma omp parallel for schedule(static) num_threads(o.nthreads)
    for (int i = 0; i < nx; ++i) {
        std::vector<Cell> col(ny);
        for (int j = 0; j < ny; ++j) col[j] = load(o.q, (size_t)j * nx + i);
        Cell lo[1], hi[1];
        ghosts(o, 1, i, col.data(), ny, 1, o.t, lo, hi);
        Z(z2, i, -1) = lo[0].q[1] / lo[0].q[0]; Z(z3, i, -1) = lo[0].q[2] / lo[0].q[0];
        Z(z2, i, ny) = hi[0].q[1] / hi[0].q[0]; Z(z3, i, ny) = hi[0].q[2] / hi[0].q[0];
    }
#pragma omp parallel for schedule(static) num_threads(o.nthreads)
    for (int j = 0; j < ny; ++j) {
        for (int i = 0; i < nx; ++i) {
            const size_t idx = (size_t)j * nx + i;
            const double lx2 = Z(z2, i + 1, j) - 2.0 * Z(z2, i, j) + Z(z2, i - 1, j);
            const double ly2 = Z(z2, i, j + 1) - 2.0 * Z(z2, i, j) + Z(z2, i, j - 1);
            const double lx3 = Z(z3, i + 1, j) - 2.0 * Z(z3, i, j) + Z(z3, i - 1, j);
            const double ly3 = Z(z3, i, j + 1) - 2.0 * Z(z3, i, j) + Z(z3, i, j - 1);
            o.q[1][idx] = o.q[1][idx] + kx * lx2 + ky * ly2;
            o.q[2][idx] = o.q[2][idx] + kx * lx3 + ky * ly3;
        }
    }
}

}  // namespace

// ===========================================================================
extern "C" {

struct orc_medium { double c0, rho0, beta, delta; };
struct orc_source { int shape; double amp, freq_hz, focus_m, centre_m, half_aperture_m, t0_s, steep, theta; };

void* orc_create(int nx, int ny, double dx, double dy, const orc_medium* m) {
    if (nx < 4 || ny < 4 || !(dx > 0) || !(dy > 0) || !m || !(m->c0 > 0) || !(m->rho0 > 0) || !(m->beta >= 1) || !(m->delta >= 0))
        return nullptr;
    Oracle* o = new Oracle();
    o->nx = nx; o->ny = ny; o->dx = dx; o->dy = dy;
    o->c0 = m->c0; o->rho0 = m->rho0; o->beta = m->beta; o->delta = m->delta;
    for (int s = 0; s < 4; ++s) { o->bc[s] = BC_EXTRAP; std::memset(&o->src[s], 0, sizeof(Source)); }
    for (int k = 0; k < 3; ++k) o->q[k].assign((size_t)nx * ny, k == 0 ? 1.0 : 0.0);
    o->t = 0.0; o->M_prev = 0.0; o->last_dt = 0.0; o->last_cfl = 0.0; o->steps = 0; o->flags = 0;
    o->x_origin = 0.0;
    o->nthreads = 1;
    return o;
}

void orc_destroy(void* h) { delete static_cast<Oracle*>(h); }

int orc_set_threads(void* h, int n) {
    Oracle* o = static_cast<Oracle*>(h);
#ifdef _OPENMP
    if (n <= 0) n = omp_get_max_threads();
#else
    n = 1;
#endif
    o->nthreads = n;
    return n;
}

int orc_set_bc(void* h, int side, int kind, const orc_source* s) {
    Oracle* o = static_cast<Oracle*>(h);
    if (side < 0 || side > 3 || kind < 0 || kind > 3) return ORC_EARG;
    if (kind == BC_SOURCE) {
        if (!s) return ORC_EARG;
        Source& d = o->src[side];
        d.shape = s->shape; d.amp = s->amp; d.freq_hz = s->freq_hz; d.focus_m = s->focus_m; d.centre_m = s->centre_m;
        d.half_aperture_m = s->half_aperture_m; d.t0_s = s->t0_s; d.steep = s->steep; d.theta = s->theta;
    }
    o->bc[side] = kind;
    return ORC_OK;
}

int orc_set_state(void* h, const double* q1, const double* q2, const double* q3) {
    Oracle* o = static_cast<Oracle*>(h);
    const size_t n = (size_t)o->nx * o->ny;
    std::copy(q1, q1 + n, o->q[0].begin());
    std::copy(q2, q2 + n, o->q[1].begin());
    std::copy(q3, q3 + n, o->q[2].begin());
    o->M_prev = 0.0; o->flags = 0;
    return ORC_OK;
}

int orc_get_state(void* h, double* q1, double* q2, double* q3) {
    Oracle* o = static_cast<Oracle*>(h);
    std::copy(o->q[0].begin(), o->q[0].end(), q1);
    std::copy(o->q[1].begin(), o->q[1].end(), q2);
    std::copy(o->q[2].begin(), o->q[2].end(), q3);
    return ORC_OK;
}

int orc_set_clock(void* h, double t_s, double last_M) {
    Oracle* o = static_cast<Oracle*>(h);
    o->t = t_s; o->M_prev = last_M > 0.0 ? last_M : 0.0;
    return ORC_OK;
}

int orc_get_info(void* h, double* t_s, double* last_dt, double* last_cfl, double* last_M, long* steps) {
    Oracle* o = static_cast<Oracle*>(h);
    if (t_s) *t_s = o->t;
    if (last_dt) *last_dt = o->last_dt;
    if (last_cfl) *last_cfl = o->last_cfl;
    if (last_M) *last_M = o->M_prev;
    if (steps) *steps = o->steps;
    return ORC_OK;
}

// O1..O5.  mode 0: value = dt [s];  mode 1: value = nu_W, dt_n = nu_W / (c0 M_{n-1})  (reading A7).
// stages: bit0 x-sweep, bit1 y-sweep, bit2 source step (7 = the full step; sub-sets exist for the pins).
int orc_step_stages(void* h, long nsteps, double value, int mode, int stages) {
    Oracle* o = static_cast<Oracle*>(h);
    if (nsteps < 0 || !(value > 0.0) || (mode != 0 && mode != 1)) return ORC_EARG;
    for (int ax = 0; ax < 2; ++ax)
        if ((o->bc[2 * ax] == BC_PERIODIC) != (o->bc[2 * ax + 1] == BC_PERIODIC)) return ORC_EARG;
    for (long n = 0; n < nsteps; ++n) {
        if (mode == 1 && !(o->M_prev > 0.0)) o->M_prev = prepass(*o);          // O7 (first step)
        const double dt = (mode == 1) ? value / (o->c0 * o->M_prev) : value;   // O1
        const double kappa = o->delta * dt / (o->dx * o->dx) + o->delta * dt / (o->dy * o->dy);
        if (kappa > 0.5) { if (mode == 0) return ORC_EARG; o->flags |= ORC_ECFL; }
        const double M = sweeps(*o, dt, stages);                              // O2, O3  Q^n -> Q* -> Q**
        if (stages & 4) source_step(*o, dt);                                   // O4  Q** -> Q^{n+1}
        o->last_dt = dt;                                                       // O5
        o->last_cfl = o->c0 * dt * M;
        if (o->last_cfl > 1.0) o->flags |= ORC_ECFL;
        o->M_prev = M;
        o->t += dt;
        o->steps += 1;
    }
    return o->flags;
}

int orc_step(void* h, long nsteps, double value, int mode) { return orc_step_stages(h, nsteps, value, mode, 7); }

// ---- unit-level entry points used by the pins ------------------------------
void orc_flux(const double q[3], double beta, int dir, double f[3]) { flux(q, beta, dir, f); }

// out: s[3], W[9] (W[p*3+m]), amdq[3], apdq[3]; returns flag
int orc_riemann(const double QL[3], const double QR[3], double beta, double* s, double* W, double* amdq, double* apdq) {
    Riemann R;
    riemann(QL, QR, beta, R);
    for (int p = 0; p < 3; ++p) { s[p] = R.s[p]; amdq[p] = R.amdq[p]; apdq[p] = R.apdq[p]; for (int m = 0; m < 3; ++m) W[p * 3 + m] = R.W[p][m]; }
    return R.flag;
}

double orc_mc_phi(double theta) { return mc_phi(theta); }

// cells: (n+4)*3 doubles, cell-major (q1,q2,q3 per cell), 2 ghosts each side; out: n*3.
int orc_sweep_line(int n, const double* cells, double lam, double beta, double* out, double* smax) {
    std::vector<Cell> c(n + 4), r(n);
    for (int k = 0; k < n + 4; ++k) for (int m = 0; m < 3; ++m) c[k].q[m] = cells[3 * k + m];
    int flag = 0; double sm = 0.0;
    sweep(n, c.data(), lam, beta, r.data(), &sm, &flag);
    for (int k = 0; k < n; ++k) for (int m = 0; m < 3; ++m) out[3 * k + m] = r[k].q[m];
    *smax = sm;
    return flag;
}

// Second stage of PAPER.md:287: "the domain moves with the propagation wave".  Move the domain by k cells in +x: the
// state is re-indexed, Q_new(i, j) = Q_old(i + k, j), the k columns that enter on the right are the x-hi ghost cells of the
// old state by the x-hi rule at the current time (zero-order extrapolation, or the analytic profile (41) at their own
// centres), and the frame of (41) moves along (x_origin).  The clock (t, lagged M) is untouched.
int orc_shift(void* h, int k) {
    Oracle* o = static_cast<Oracle*>(h);
    if (k < 0 || k >= o->nx) return ORC_EARG;
    if (o->bc[SIDE_XLO] == BC_PERIODIC || o->bc[SIDE_XHI] == BC_PERIODIC || o->bc[SIDE_XHI] == BC_REFLECT) return ORC_EARG;
    if (k == 0) return ORC_OK;
    const int nx = o->nx, ny = o->ny;
    std::vector<Cell> row(nx), lo(k), hi(k);
    for (int j = 0; j < ny; ++j) {
        for (int i = 0; i < nx; ++i) row[i] = load(o->q, (size_t)j * nx + i);
        ghosts(*o, 0, j, row.data(), nx, k, o->t, lo.data(), hi.data());
        for (int i = 0; i < nx; ++i) {
            const Cell& c = (i + k < nx) ? row[i + k] : hi[i + k - nx];
            for (int m = 0; m < 3; ++m) o->q[m][(size_t)j * nx + i] = c.q[m];
        }
    }
    o->x_origin += k * o->dx;
    return ORC_OK;
}

// boundary source cell as the ghost rule evaluates it (for tests of (41)/(43))
int orc_source_cell(void* h, int side, double along_m, double xc_m, double yc_m, double t, double out[3]) {
    Oracle* o = static_cast<Oracle*>(h);
    Cell c;
    const bool in = source_cell(*o, side, along_m, xc_m, yc_m, t, &c);
    if (in) { out[0] = c.q[0]; out[1] = c.q[1]; out[2] = c.q[2]; }
    return in ? 1 : 0;
}

double orc_prepass(void* h) { return prepass(*static_cast<Oracle*>(h)); }

}  // extern "C"
