// fvnl_fused.cuh -- the one-pass step kernel: x-sweep (24), y-sweep (25) and source step (26) of arXiv 1311.3004
// in ONE pass over the state, every Riemann problem solved once.
//
// Mapping.  A thread block owns a strip of BX consecutive columns (BX-6 of them produce output: the per-step
// dependency cone is 3 cells wide) and marches over a chunk of rows.  One thread = one column.
// Row r of Q^n enters at "tick" r and moves through a software pipeline held in registers:
//     tick r :  Q^n(.,r) --x-Riemann, x-flux--> Q*(.,r)                       neighbours in x: shared memory
//               Q*(.,r-1), Q*(.,r) --y-Riemann--> Wy(r-1/2)                   neighbours in y: this thread, earlier ticks
//               Wy(r-5/2), Wy(r-3/2), Wy(r-1/2) --y-flux--> Q**(.,r-2)
//               Q**(.,r-4), Q**(.,r-3), Q**(.,r-2) --source step--> Q^{n+1}(.,r-3) --> HBM
// so each state array is read once and written once per time step (plus the 3-cell halos of strips and chunks);
// waves, fluctuations and the intermediate states Q*, Q** never touch HBM (PAPER.md:159-198 quantities live in
// registers; the x-neighbour exchange goes through 17 doubles of shared memory per column).
//
// Ghost cells (readings A9, A10, A14 of DESIGN.md) are evaluated on load: the x rule maps the thread's column once,
// the y rule maps the row of each tick; the one-deep ghosts of Q** that the source step needs are derived from the
// neighbouring interior Q** at the edge columns / rows.
#pragma once
#include "fvnl_unfused.cuh"

namespace fvnl {

// Per-thread description of its column after the x rule (fixed for the whole march).
struct ColMap {
    int col;        // column to load from (wrapped / clamped / mirrored)
    bool neg2;      // REFLECT ghost column: normal momentum negated
    int xsrc;       // side index (SIDE_XLO / SIDE_XHI) if the column is a ghost of a SOURCE side, else -1
};

__device__ __forceinline__ ColMap map_column(const Grid& g, int i) {
    ColMap m;
    m.col = i; m.neg2 = false; m.xsrc = -1;
    if (i < 0 || i >= g.nx) {
        const int sd = i < 0 ? SIDE_XLO : SIDE_XHI;
        const int kind = g.side[sd].kind;
        if (kind == BC_PERIODIC) m.col = wrap(i, g.nx);
        else if (kind == BC_REFLECT) { m.col = clampi(i < 0 ? -1 - i : 2 * g.nx - 1 - i, g.nx); m.neg2 = true; }
        else { m.col = clampi(i, g.nx); if (kind == BC_SOURCE) m.xsrc = sd; }
    }
    return m;
}

// Row of the ghost-extended mesh -> row to load from, by the y rule (block-uniform).
struct RowMap {
    int row;
    bool neg3;
    int ysrc;       // SIDE_YLO / SIDE_YHI if the row is a ghost of a SOURCE side, else -1
};

__device__ __forceinline__ RowMap map_row(const Grid& g, int r) {
    RowMap m;
    m.row = r; m.neg3 = false; m.ysrc = -1;
    if (r < 0 || r >= g.ny) {
        const int sd = r < 0 ? SIDE_YLO : SIDE_YHI;
        const int kind = g.side[sd].kind;
        if (kind == BC_PERIODIC) m.row = wrap(r, g.ny);
        else if (kind == BC_REFLECT) { m.row = clampi(r < 0 ? -1 - r : 2 * g.ny - 1 - r, g.ny); m.neg3 = true; }
        else { m.row = clampi(r, g.ny); if (kind == BC_SOURCE) m.ysrc = sd; }
    }
    return m;
}

// Analytic override of a loaded ghost value (same precedence as load_ext: x rule first, then y rule).
__device__ __noinline__ void apply_sources(const Grid& g, const ColMap& cm, const RowMap& rm, int i, int r, double t,
                                           Q3& c) {
    if (cm.xsrc >= 0) {
        Q3 s;
        if (source_cell(g.side[cm.xsrc], cm.xsrc, g.c0, (r + 0.5) * g.dy, (i + 0.5) * g.dx, t, s)) { c = s; return; }
    }
    if (rm.ysrc >= 0) {
        Q3 s;
        const double x = (cm.col + 0.5) * g.dx;                 // the (x-mapped) column the y rule is applied on
        if (source_cell(g.side[rm.ysrc], rm.ysrc, g.c0, x, x, t, s)) {
            if (cm.neg2) s.q2 = -s.q2;
            c = s;
        }
    }
}

// z = (q2/q1, q3/q1) of the one-deep ghost of an intermediate state (source step, reading A9).
__device__ __noinline__ void ghost_z(const Grid& g, int sd, const Q3& inner, double along, double xc, double t,
                                     double& z2, double& z3) {
    const Q3 c = ghost_of(g, sd, inner, along, xc, t);
    const double rc = rcp_o1(c.q1);
    z2 = c.q2 * rc;
    z3 = c.q3 * rc;
}

struct WaveLite {                 // what a neighbouring interface contributes to the limiter
    double al1, s1, r31, al2, s2, r32, al3;
};

// The step kernel.  grid = (strips, chunks); block = BX threads.  rows: rows of output per chunk.
template <int BX>
__global__ void __launch_bounds__(BX) k_step_fused(Grid g, Clock* clk, const double* __restrict__ q1,
                                                   const double* __restrict__ q2, const double* __restrict__ q3,
                                                   double* __restrict__ o1, double* __restrict__ o2,
                                                   double* __restrict__ o3, int rows) {
    __shared__ double s_cell[5][BX];      // q1 q2 q3 hz2 hz3 of the cell of this column          (tick r)
    __shared__ double s_wave[7][BX];      // al1 s1 r31 al2 s2 r32 al3 of the interface i-1/2      (tick r)
    __shared__ double s_gm[3][BX];        // left-going part of the interface i-1/2                (tick r)
    __shared__ double s_z[2][BX];         // q2/q1, q3/q1 of Q**                                   (row r-2)

    const int tid = threadIdx.x;
    const int i = (int)blockIdx.x * (BX - 6) - 3 + tid;            // column on the ghost-extended mesh
    const int j0 = (int)blockIdx.y * rows;
    const int j1 = min(j0 + rows, g.ny);
    const double t = clk->t, lamx = clk->lamx, lamy = clk->lamy, kapx = clk->kapx, kapy = clk->kapy;
    const double b2 = 2.0 * (g.beta - 1.0);
    const bool px = g.side[SIDE_XLO].kind == BC_PERIODIC, py = g.side[SIDE_YLO].kind == BC_PERIODIC;
    const bool any_src = g.side[0].kind == BC_SOURCE || g.side[1].kind == BC_SOURCE || g.side[2].kind == BC_SOURCE ||
                         g.side[3].kind == BC_SOURCE;

    const ColMap cm = map_column(g, i);
    const int tl = tid > 0 ? tid - 1 : 0, tr = tid < BX - 1 ? tid + 1 : BX - 1;
    // which results of this thread are real
    const bool x_if_m = tid >= 1 && i >= 0 && i <= g.nx;           // interface i-1/2 enters M (touches an interior cell)
    const bool x_if_f = tid >= 1 && i >= -1 && i <= g.nx + 1;      // interface i-1/2 is one the scheme solves
    const bool y_col = tid >= 2 && tid <= BX - 3 && i >= 0 && i < g.nx;   // Q* of this column is valid and interior
    const bool out_col = tid >= 3 && tid <= BX - 4 && i >= 0 && i < g.nx;
    const bool fixW = !px && i == 0, fixE = !px && i == g.nx - 1;

    int flags = 0;
    double smx = 0.0, smy = 0.0;

    // rolling state (all in y-form where noted: components 2 and 3 switched)
    CellX cyA = {1.0, 0.0, 0.0, 0.0, 0.0};                        // y-cell of Q*(r-1)
    double sB1 = 1.0, sB2 = 0.0, sB3 = 0.0;                        // Q*(r-2), y-form
    Waves wA = {0, 1, 0, 0, -1, 0, 0, 0}, wB = wA;                 // Wy(r-3/2), Wy(r-5/2)
    double gB1 = 0.0, gB2 = 0.0, gB3 = 0.0;                        // right-going part of the y-interface r-5/2
    double c1 = 1.0, c2 = 0.0, c3 = 0.0, zC2 = 0.0, zC3 = 0.0, lC2 = 0.0, lC3 = 0.0;   // Q**(r-3), its z and d2x z
    double zS2 = 0.0, zS3 = 0.0;                                   // z of Q**(r-4)

    // first row
    int r = j0 - 3;
    RowMap rm = map_row(g, r);
    size_t idx = (size_t)rm.row * g.nx + cm.col;
    Q3 nxt;
    nxt.q1 = q1[idx]; nxt.q2 = q2[idx]; nxt.q3 = q3[idx];

    for (; r < j1 + 3; ++r) {
        // ---- this tick's cell; prefetch the next row --------------------------------------------------------
        Q3 q = nxt;
        if (cm.neg2) q.q2 = -q.q2;
        if (rm.neg3) q.q3 = -q.q3;
        if (any_src && (cm.xsrc >= 0 || rm.ysrc >= 0)) apply_sources(g, cm, rm, i, r, t, q);
        const RowMap rm_next = map_row(g, r + 1);
        idx = (size_t)rm_next.row * g.nx + cm.col;
        nxt.q1 = q1[idx]; nxt.q2 = q2[idx]; nxt.q3 = q3[idx];
        const bool row_in = r >= 0 && r < g.ny;

        // ---- x-sweep of row r (27)-(30) ---------------------------------------------------------------------
        int fx = 0;
        const CellX cx = make_cell(q.q1, q.q2, q.q3, fx);
        s_cell[0][tid] = cx.q1; s_cell[1][tid] = cx.q2; s_cell[2][tid] = cx.q3; s_cell[3][tid] = cx.hz2; s_cell[4][tid] = cx.hz3;
        __syncthreads();
        CellX L;
        L.q1 = s_cell[0][tl]; L.q2 = s_cell[1][tl]; L.q3 = s_cell[2][tl]; L.hz2 = s_cell[3][tl]; L.hz3 = s_cell[4][tl];
        const Waves w = riemann_x(L, cx, b2, fx);
        s_wave[0][tid] = w.al1; s_wave[1][tid] = w.s1; s_wave[2][tid] = w.r31; s_wave[3][tid] = w.al2;
        s_wave[4][tid] = w.s2; s_wave[5][tid] = w.r32; s_wave[6][tid] = w.al3;
        __syncthreads();
        Flux3 F;
        {
            const int u1 = w.s1 > 0.0 ? tl : tr, u2 = w.s2 > 0.0 ? tl : tr, u3 = w.s3 > 0.0 ? tl : tr;
            F = interface_flux(w, s_wave[0][u1], s_wave[1][u1], s_wave[2][u1], s_wave[3][u2], s_wave[4][u2],
                               s_wave[5][u2], s_wave[6][u3], lamx);
        }
        s_gm[0][tid] = F.m1; s_gm[1][tid] = F.m2; s_gm[2][tid] = F.m3;
        if (row_in) {
            if (x_if_m) smx = fmax(smx, max_speed(w));
            if (x_if_f) flags |= fx;
        }
        __syncthreads();
        Q3 st;                                                    // Q*(i, r)
        st.q1 = fma(-lamx, F.p1 + s_gm[0][tr], q.q1);
        st.q2 = fma(-lamx, F.p2 + s_gm[1][tr], q.q2);
        st.q3 = fma(-lamx, F.p3 + s_gm[2][tr], q.q3);
        if (row_in && y_col && (not_finite(st.q1) || not_finite(st.q2) || not_finite(st.q3))) flags |= F_ENAN;

        // ---- y-sweep: interface r-1/2, flux of interface r-3/2, Q**(r-2) -------------------------------------
        int fy = 0;
        const CellX cyN = make_cell(st.q1, st.q3, st.q2, fy);
        const Waves wN = riemann_x(cyA, cyN, b2, fy);
        Flux3 G;
        {
            const bool u1 = wA.s1 > 0.0, u2 = wA.s2 > 0.0, u3 = wA.s3 > 0.0;
            G = interface_flux(wA, u1 ? wB.al1 : wN.al1, u1 ? wB.s1 : wN.s1, u1 ? wB.r31 : wN.r31,
                               u2 ? wB.al2 : wN.al2, u2 ? wB.s2 : wN.s2, u2 ? wB.r32 : wN.r32,
                               u3 ? wB.al3 : wN.al3, lamy);
        }
        Q3 n;                                                     // Q**(i, r-2), physical component order
        n.q1 = fma(-lamy, gB1 + G.m1, sB1);
        n.q3 = fma(-lamy, gB2 + G.m2, sB2);
        n.q2 = fma(-lamy, gB3 + G.m3, sB3);
        if (y_col && r >= j0 - 2 && r >= -1 && r <= g.ny + 1) {   // interface r-1/2 is one the scheme solves
            flags |= fy;
            if (r >= 0 && r <= g.ny) smy = fmax(smy, max_speed(wN));
        }
        if (y_col && r >= j0 + 1 && r - 2 >= 0 && r - 2 < g.ny &&
            (not_finite(n.q1) || not_finite(n.q2) || not_finite(n.q3))) flags |= F_ENAN;
        gB1 = G.p1; gB2 = G.p2; gB3 = G.p3;
        wB = wA; wA = wN;
        sB1 = cyA.q1; sB2 = cyA.q2; sB3 = cyA.q3;
        cyA = cyN;

        // ---- source step (26): d2x z of row r-2 now, output row R = r-3 ---------------------------------------
        const double rn = rcp_o1(n.q1);
        const double zN2 = n.q2 * rn, zN3 = n.q3 * rn;
        s_z[0][tid] = zN2; s_z[1][tid] = zN3;
        __syncthreads();
        double zW2 = s_z[0][tl], zW3 = s_z[1][tl], zE2 = s_z[0][tr], zE3 = s_z[1][tr];
        if (fixW) ghost_z(g, SIDE_XLO, n, (r - 2 + 0.5) * g.dy, -0.5 * g.dx, t, zW2, zW3);
        if (fixE) ghost_z(g, SIDE_XHI, n, (r - 2 + 0.5) * g.dy, (g.nx + 0.5) * g.dx, t, zE2, zE3);
        const double lN2 = (zE2 + zW2) - 2.0 * zN2, lN3 = (zE3 + zW3) - 2.0 * zN3;
        const int R = r - 3;
        if (R >= j0) {                                            // R < j1 by the loop bound
            double a2 = zS2, a3 = zS3, b2n = zN2, b3n = zN3;
            if (!py) {
                Q3 c; c.q1 = c1; c.q2 = c2; c.q3 = c3;
                const double x = (i + 0.5) * g.dx;
                if (R == 0) ghost_z(g, SIDE_YLO, c, x, x, t, a2, a3);
                if (R == g.ny - 1) ghost_z(g, SIDE_YHI, c, x, x, t, b2n, b3n);
            }
            const double ly2 = (b2n + a2) - 2.0 * zC2, ly3 = (b3n + a3) - 2.0 * zC3;
            if (out_col) {
                const size_t o = (size_t)R * g.nx + i;
                o1[o] = c1;
                o2[o] = fma(kapy, ly2, fma(kapx, lC2, c2));
                o3[o] = fma(kapy, ly3, fma(kapx, lC3, c3));
            }
        }
        zS2 = zC2; zS3 = zC3;
        c1 = n.q1; c2 = n.q2; c3 = n.q3; zC2 = zN2; zC3 = zN3; lC2 = lN2; lC3 = lN3;
        rm = rm_next;
    }
    block_max_to(&clk->sx_bits, smx);
    __syncthreads();
    block_max_to(&clk->sy_bits, smy);
    block_flags_to(&clk->flags, flags);
}

}  // namespace fvnl
