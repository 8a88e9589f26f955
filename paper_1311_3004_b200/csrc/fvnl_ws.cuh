// fvnl_ws.cuh -- the one-pass step kernel, warp specialised: half of a block's warps run the x-sweep, the other half
// the y-sweep and the source step, on the same strip of columns.
//
// Why.  The fused kernel (fvnl_fused.cuh) carries the whole rolling state of a column in one thread: ~168 registers,
// 12 warps per SM, and since a warp issues in order and a dependent FP64 operation waits 9 cycles (measured), the
// FP64 pipe sits half idle (profiles/).  The x-sweep of a row needs NO state from earlier rows; the y-sweep needs the
// rolling window.  Splitting the two gives x-warps a small register footprint and y-warps a medium one
// (setmaxnreg moves registers from the first to the second), 16 warps per SM instead of 12, and two independent
// instruction streams per scheduler that never wait on each other's barriers except once per tick:
//     tick r, X warps :  Q^n(., r) -> cells -> [bar X] -> Riemann solves -> [bar X] -> limited fluxes
//                        -> publish  u = Q^n - lam_x G+  and  G-  of row r (parity r&1)            -> [bar ALL]
//     tick r, Y warps :  Q*(., r-1) = u - lam_x G-(right neighbour)  (published in tick r-1)
//                        -> y-Riemann solve, limited y-flux -> Q**(., r-3) -> source step -> Q^{n+1}(., r-4) -> HBM
//                        -> publish z of Q** for the neighbours' source step (parity r&1)        -> [bar ALL]
// Arithmetic, ghost rules and validity masks are those of fvnl_fused.cuh.
//
// Analytic SOURCE edges: the ghost cells of the step are computed beforehand by the boundary kernel k_sources
// (fvnl.cu) into Grid::src and only LOADED here (ptxas 12.9 crashes on setmaxnreg in a kernel that also calls the
// out-of-line sin / exp / tanh paths, and evaluating them inside the march made the strip that owns the edge twice as
// slow as the others).
#pragma once
#include "fvnl_fused.cuh"

namespace fvnl {

constexpr int WS_COLS = 128;                  // columns of a strip = threads of each group
// shared memory (bytes): arrays of double2, WS_COLS + 2 elements each, ALL double-buffered by the parity of the row they hold
//   X group:  0 (q1,q2)  1 (q3,hz2)  2 (hz3,-)  [cells]      3 (al1,s1)  4 (r31,al3)  5 (al2,s2)  6 (r32,-)  [waves]
//   X -> Y:   7 (m1,m2)  8 (m3,ft1)  9 (u1,u2)  10 (u3,p1)       Y -> Y:  11 (z2,z3)
constexpr int WS_ARRAYS = 12;
__host__ __device__ constexpr int ws_arr2(int k, int parity) { return (2 * k + parity) * (WS_COLS + 2) * 16; }
__host__ __device__ constexpr int ws_ring_off() { return 2 * WS_ARRAYS * (WS_COLS + 2) * 16; }
__host__ __device__ constexpr int ws_smem_bytes() { return ws_ring_off() + 4 * 3 * WS_COLS * 8; }

__device__ __forceinline__ void bar_x() { asm volatile("bar.sync 1, 128;" ::: "memory"); }
__device__ __forceinline__ void bar_all() { asm volatile("bar.sync 2, 256;" ::: "memory"); }

struct XThread {
    ColMap cm;
    int i, special;
    char *p, *pq;
    double smx;
    int mqx, mdx;
    Wv w;                                    // waves of interface i-1/2 of the row solved in the previous tick
    double rn1, rn2;                         // and their 1/(r.r)
    Cx cx;                                   // this column's cell of the row converted in the previous tick
    double aq[2][3];                         // Q^n(i, .) of the rows loaded in the previous two ticks, by row parity
};

// One tick of an X warp.  The x-sweep is software-pipelined over rows: tick t runs three INDEPENDENT pieces of work, each on
// its own row, so that the warp has several dependency chains to issue from (a dependent FP64 operation waits 9 cycles) and
// ONE block-wide barrier per tick separates everything:
//   phase C, row t   : limited fluxes (28)-(30) of interface i-1/2 from its waves (solved in tick t-1, kept in registers)
//                      and the upwind neighbour's (shared memory) -> the two halves of the update (27) for the Y warps;
//   phase B, row t+1 : Riemann solve between the cells of columns i-1 and i (converted in tick t-1)
//                      -> waves to shared memory;
//   phase A, row t+2 : Q^n(., t+2) from the prefetch ring, ghost rule, primitive conversion -> cell to shared memory;
//                      prefetch of row t+4.
// P = t & 1.  FILL: one of the two ticks before the Y warps start (the barrier is then the X group's own).
template <int P, bool STEADY>
__device__ __forceinline__ void ws_xtick(const Grid& g, const StepK& k, XThread& th, int t, int r0,
                                         const double* __restrict__ q1, const double* __restrict__ q2,
                                         const double* __restrict__ q3) {
    char* const p = th.p;
    constexpr int Q = P ^ 1;
    // ---- phase C: row t ----------------------------------------------------------------------------------------------
    if (STEADY || t >= r0) {
        const Wv& w = th.w;
        const char* u1 = p + (hi_word(w.s1) < 0 ? 16 : -16);                  // upwind interface
        const char* u2 = p + (hi_word(w.s2) < 0 ? 16 : -16);
        const char* u3 = p + (hi_word(w.v) < 0 ? 16 : -16);
        const double2 k1 = lds2(u1 + ws_arr2(3, P)), k2 = lds2(u2 + ws_arr2(5, P));
        const double k1r = lds1(u1 + ws_arr2(4, P)), k2r = lds1(u2 + ws_arr2(6, P)), k3 = lds1(u3 + ws_arr2(4, P) + 8);
        const double own1 = th.aq[P][0], own2 = th.aq[P][1], a3 = th.aq[P][2];   // Q^n(i, t), loaded two ticks ago
        const double b1 = k1.x * rdot(k1.y, k1r, w.s1, w.r31) * th.rn1;
        const double b2 = k2.x * rdot(k2.y, k2r, w.s2, w.r32) * th.rn2;
        const Fl F = flux2(w, b1, b2, k3, k.lamx);
        // the two halves of (27) for row t: what this interface sends left, and this column's own part
        // (the density component goes over unrounded: q1, p1 and the first component of F~, see update_q1)
        sts2(p + ws_arr2(7, P), F.m1, F.m2); sts2(p + ws_arr2(8, P), F.m3, F.ft1);
        sts2(p + ws_arr2(9, P), own1, fma(-k.lamx, F.p2, own2));
        sts2(p + ws_arr2(10, P), fma(-k.lamx, F.p3, a3), F.p1);
    }
    // ---- phase B: row t+1 --------------------------------------------------------------------------------------------
    if (STEADY || t + 1 >= r0) {
        Cx L;
        const Cx C = th.cx;
        {
            const double2 l0 = lds2(p + ws_arr2(0, Q) - 16), l1 = lds2(p + ws_arr2(1, Q) - 16);
            L.q1 = l0.x; L.q2 = l0.y; L.q3 = l1.x; L.hz2 = l1.y; L.hz3 = lds1(p + ws_arr2(2, Q) - 16);
        }
        int td = 0x7fffffff;
        const Wv w = riemann2(L, C, k.b2, k.omb2, td);
        th.rn1 = rnorm(w.s1, w.r31); th.rn2 = rnorm(w.s2, w.r32);
        th.w = w;
        sts2(p + ws_arr2(3, Q), w.al1, w.s1); sts2(p + ws_arr2(4, Q), w.r31, w.al3); sts2(p + ws_arr2(5, Q), w.al2, w.s2);
        sts1(p + ws_arr2(6, Q), w.r32);
        if (STEADY || (unsigned)(t + 1) < (unsigned)g.ny) {
            th.mdx = min(th.mdx, td);
            th.smx = dmax(th.smx, fabs(hi_word(w.v) < 0 ? w.s2 : w.s1));      // max(|s1|,|s2|) = |v| + a
        }
    }
    // ---- phase A: row t+2 (prefetch row t+4) -------------------------------------------------------------------------
    {
        const int r = t + 2;
        RowMap rm, rm_pre;
        if (STEADY) {
            rm.row = r; rm.neg3 = false; rm.ysrc = -1;
            rm_pre.row = r + 2;
        } else {
            rm = map_row(g, r);
            rm_pre = map_row(g, r + 2);
        }
        cp_async_wait<1>();                                                   // row t+2 has landed
        double a1, a2, a3;
        {
            const char* ps = th.pq + (r & 3) * (3 * WS_COLS * 8);
            a1 = lds1(ps); a2 = lds1(ps + WS_COLS * 8); a3 = lds1(ps + 2 * WS_COLS * 8);
            char* pd = th.pq + ((r + 2) & 3) * (3 * WS_COLS * 8);
            const size_t idx = (size_t)rm_pre.row * g.nx + th.cm.col;
            cp_async8(pd, q1 + idx); cp_async8(pd + WS_COLS * 8, q2 + idx); cp_async8(pd + 2 * WS_COLS * 8, q3 + idx);
            cp_async_commit();
        }
        if ((th.special & 12) || (!STEADY && (rm.neg3 || rm.ysrc >= 0))) {    // ghost column / row with a rule: rare
            if (!STEADY && rm.neg3) a3 = -a3;
            if (th.special & 4) a2 = -a2;
            bool done = false;                                                // x rule first, then y rule (as load_mapped)
            if ((th.special & 8) && r >= -3 && r <= g.ny + 2) {
                const int sd = th.cm.xsrc, l = sd == SIDE_XLO ? -1 - th.i : th.i - g.nx;
                if (l < 3) {
                    const double* sp = k.src + src_off(g.nx, g.ny, sd) + 3 * ((size_t)(g.ny + 6) * l + r + 3);
                    if (sp[0] > 0.0) { a1 = sp[0]; a2 = sp[1]; a3 = sp[2]; done = true; }
                }
            }
            if (!STEADY && !done && rm.ysrc >= 0) {
                const int sd = rm.ysrc, l = sd == SIDE_YLO ? -1 - r : r - g.ny;
                if (l < 3) {
                    const double* sp = k.src + src_off(g.nx, g.ny, sd) + 3 * ((size_t)g.nx * l + th.cm.col);
                    if (sp[0] > 0.0) { a1 = sp[0]; a2 = th.cm.neg2 ? -sp[1] : sp[1]; a3 = sp[2]; }
                }
            }
        }
        int tq = 0x7fffffff;
        const Cx cx = cell_of(a1, a2, a3, tq);
        sts2(p + ws_arr2(0, P), cx.q1, cx.q2); sts2(p + ws_arr2(1, P), cx.q3, cx.hz2); sts1(p + ws_arr2(2, P), cx.hz3);
        th.cx = cx;
        th.aq[P][0] = a1; th.aq[P][1] = a2; th.aq[P][2] = a3;
        if (STEADY || (unsigned)r < (unsigned)g.ny) th.mqx = min(th.mqx, tq);
    }
    if (!STEADY && t < r0) bar_x(); else bar_all();                           // the Y warps join at tick r0
}

// z of the one-deep ghost of Q** at a non-periodic edge, from the z of the interior cell next to it (reading A9): EXTRAP
// copies, REFLECT negates the normal velocity, SOURCE takes the analytic cell of layer 0 (record `m`: the row for an x
// side, the column for a y side) if it lies inside the aperture.
__device__ __forceinline__ double2 ghost_z_plain(const Grid& g, const double* __restrict__ src, int sd, int m, double z2, double z3) {
    const int kind = g.side[sd].kind;
    if (kind == BC_REFLECT) return sd < 2 ? make_double2(-z2, z3) : make_double2(z2, -z3);
    if (kind == BC_SOURCE) {
        m = sd < 2 ? min(max(m, -3), g.ny + 2) : min(max(m, 0), g.nx - 1);          // (halo threads / pipeline fill: value unused)
        const double* sp = src + src_off(g.nx, g.ny, sd) + 3 * (size_t)(sd < 2 ? m + 3 : m);
        if (sp[0] > 0.0) {
            const double rc = rcp_o1(sp[0]);
            return make_double2(sp[1] * rc, sp[2] * rc);
        }
    }
    return make_double2(z2, z3);
}

struct YThread {
    int i, special;
    bool out_col;
    char* p;
    double smy;
    int mqy, mdy, mxo;
};

struct YCarry {
    double gp1, gp2, gp3, gf1;               // right-going part (and F~, comp. 1) of the y-interface below B
    double q1, q2, q3;                       // Q*(., ry-4), y-form
    double c1, c2, c3, zC2, zC3;             // Q**(ry-5) and its z
    double zS2, zS3;                         // z of Q**(ry-6)
    Cx pend;                                 // cell of Q*(., ry-1), y-form: converted in the previous tick, solved in this one
};

// One tick of a Y warp (tick r works on ry = r-1, the row the X warps published in the previous tick).  I(k) = the
// y-interface between rows k-1 and k.  THREE independent chains per tick -- the y-sweep is software-pipelined over rows so
// that the warp always has several instructions to choose from against the 9-cycle FP64 latency, and so that the longest
// dependent chain of a tick is the Riemann solve alone:
//   chain 1a:  Q*(., ry) completed from what the X warps published -> primitive conversion (cy.pend, solved next tick);
//   chain 1b:  y-Riemann solve of N = I(ry-1) from the two cells converted in earlier ticks -> limiter inputs between N
//              and A = I(ry-2), which are now final for A;
//   chain 2:   limited flux of B = I(ry-3) (its limiter inputs became final in the previous tick) -> Q**(., ry-4)
//              -> source step for row ry-5 -> Q^{n+1}(., ry-5) -> HBM.
// P = r & 1: parity this tick publishes into (it reads parity P^1); Y[P] holds B on entry and N on exit, Y[P^1] is A.
template <int P, bool STEADY>
__device__ __forceinline__ void ws_ytick(const Grid& g, const StepK& k, YThread& th, YCarry& cy, YSet& Y0, YSet& Y1, int r,
                                         double* __restrict__ o1, double* __restrict__ o2, double* __restrict__ o3) {
    YSet& N = P ? Y1 : Y0;
    YSet& A = P ? Y0 : Y1;
    constexpr int R = P ^ 1;
    char* const p = th.p;
    const int ry = r - 1;
    // ---- chain 2: flux of B, Q**(., ry-4), source step ----------------------------------------------------------------
    const Fl G = flux2(N.w, N.pb1, N.pb2, N.pb3, k.lamy);                     // N still holds B
    const double n1 = update_q1(cy.q1, k.lamy, cy.gp1 + G.m1, cy.gf1, G.ft1); // Q**(i, ry-4); physical order n1, n2, n3
    const double n3 = fma(-k.lamy, cy.gp2 + G.m2, cy.q2);
    const double n2 = fma(-k.lamy, cy.gp3 + G.m3, cy.q3);
    cy.gp1 = G.p1; cy.gp2 = G.p2; cy.gp3 = G.p3; cy.gf1 = G.ft1;
    cy.q1 = N.c.q1; cy.q2 = N.c.q2; cy.q3 = N.c.q3;                           // Q*(ry-3), y-form: next tick's lower row
    double2 zW = lds2(p + ws_arr2(11, R) - 16), zE = lds2(p + ws_arr2(11, R) + 16);   // z of row ry-5, published last tick
    if (th.special & 3) {
        if (th.special & 1) zW = ghost_z_plain(g, k.src, SIDE_XLO, ry - 5, cy.zC2, cy.zC3);
        if (th.special & 2) zE = ghost_z_plain(g, k.src, SIDE_XHI, ry - 5, cy.zC2, cy.zC3);
    }
    const double H2 = fma(k.k2, cy.zC2, fma(k.kapx, zE.x + zW.x, cy.c2));
    const double H3 = fma(k.k2, cy.zC3, fma(k.kapx, zE.y + zW.y, cy.c3));
    const double rq = rcp_o1(n1);
    const double zN2 = n2 * rq, zN3 = n3 * rq;
    sts2(p + ws_arr2(11, P), zN2, zN3);
    const int Ro = ry - 5;
    if (STEADY || Ro >= k.j0) {                                               // Ro < j1 by the loop bound
        double y2 = zN2 + cy.zS2, y3 = zN3 + cy.zS3;
        if (!STEADY && !k.py && (Ro == 0 || Ro == g.ny - 1)) {
            double2 lo = make_double2(cy.zS2, cy.zS3), hi = make_double2(zN2, zN3);
            if (Ro == 0) lo = ghost_z_plain(g, k.src, SIDE_YLO, th.i, cy.zC2, cy.zC3);
            if (Ro == g.ny - 1) hi = ghost_z_plain(g, k.src, SIDE_YHI, th.i, cy.zC2, cy.zC3);
            y2 = hi.x + lo.x; y3 = hi.y + lo.y;
        }
        const double w2 = fma(k.kapy, y2, H2), w3 = fma(k.kapy, y3, H3);
        if (th.out_col) {
            const size_t o = (size_t)Ro * g.nx + th.i;
            o1[o] = cy.c1; o2[o] = w2; o3[o] = w3;
            th.mxo = max(th.mxo, max(hi_word(cy.c1) & 0x7fffffff, max(hi_word(w2) & 0x7fffffff, hi_word(w3) & 0x7fffffff)));
        }
    }
    cy.zS2 = cy.zC2; cy.zS3 = cy.zC3;
    cy.c1 = n1; cy.c2 = n2; cy.c3 = n3; cy.zC2 = zN2; cy.zC3 = zN3;

    // ---- chain 1b: interface N = I(ry-1) between the cells of Q*(ry-2) (A.c) and Q*(ry-1) (cy.pend); limiter inputs of A ----
    int tdy = 0x7fffffff;
    N.c = cy.pend;
    N.w = riemann2(A.c, N.c, k.b2, k.omb2, tdy);
    N.rn1 = rnorm(N.w.s1, N.w.r31); N.rn2 = rnorm(N.w.s2, N.w.r32);
    const double d1 = rdot(A.w.s1, A.w.r31, N.w.s1, N.w.r31), d2 = rdot(A.w.s2, A.w.r32, N.w.s2, N.w.r32);
    N.pb1 = A.w.al1 * d1 * N.rn1; N.pb2 = A.w.al2 * d2 * N.rn2; N.pb3 = A.w.al3;      // if A is N's upwind side
    const double hb1 = N.w.al1 * d1 * A.rn1, hb2 = N.w.al2 * d2 * A.rn2;              // if N is A's upwind side
    A.pb1 = hi_word(A.w.s1) < 0 ? hb1 : A.pb1;                                // A's upwind side is now known
    A.pb2 = hi_word(A.w.s2) < 0 ? hb2 : A.pb2;
    A.pb3 = hi_word(A.w.v) < 0 ? N.w.al3 : A.pb3;
    if (STEADY || (unsigned)(ry - 1 - k.ylo) <= (unsigned)k.ycnt) {           // I(ry-1) is an interface the scheme solves
        th.mdy = min(th.mdy, tdy);
        if (STEADY || (unsigned)(ry - 1) <= (unsigned)g.ny) th.smy = dmax(th.smy, fabs(hi_word(N.w.v) < 0 ? N.w.s2 : N.w.s1));
    }

    // ---- chain 1a: Q*(., ry), the update (27) completed, and its primitive conversion for the next tick ----------------
    {
        const double2 u = lds2(p + ws_arr2(9, R)), gm = lds2(p + ws_arr2(7, R) + 16);
        const double2 u3 = lds2(p + ws_arr2(10, R)), gm3 = lds2(p + ws_arr2(8, R) + 16);
        const double ft_own = lds1(p + ws_arr2(8, R) + 8);
        const double s1 = update_q1(u.x, k.lamx, u3.y + gm.x, ft_own, gm3.y);
        const double s2 = fma(-k.lamx, gm.y, u.y), s3 = fma(-k.lamx, gm3.x, u3.x);
        int tqy = 0x7fffffff;
        cy.pend = cell_of(s1, s3, s2, tqy);                                   // positions 2,3 switched
        if (STEADY || (unsigned)(ry - k.ylo) <= (unsigned)k.ycnt) th.mqy = min(th.mqy, tqy);   // a cell the y-sweep uses
    }
    bar_all();
}

// The step kernel.  grid = (strips, chunks); block = 256 threads (warps 0-3: X group, warps 4-7: Y group);
// dynamic shared memory = ws_smem_bytes().  The kernel is compiled for 128 registers per thread (2 blocks per SM) and
// setmaxnreg moves registers from the X warps (96) to the Y warps (160).  value / mode / more: see step_tail.
constexpr int WS_BLOCKS_PER_SM = 2;
__global__ void __launch_bounds__(256, WS_BLOCKS_PER_SM)
k_step_ws(Grid g, Clock* clk, const double* __restrict__ q1, const double* __restrict__ q2,
          const double* __restrict__ q3, double* __restrict__ o1, double* __restrict__ o2, double* __restrict__ o3,
          int rows, double value, int mode, int more) {
    extern __shared__ __align__(16) char smem[];
    const int tid = threadIdx.x;
    for (int j = tid; j < ws_smem_bytes() / 8; j += 256) reinterpret_cast<double*>(smem)[j] = 1.0;   // finite fill

    StepK k;
    k.t = clk->t; k.lamx = clk->lamx; k.lamy = clk->lamy; k.kapx = clk->kapx; k.kapy = clk->kapy;
    k.k2 = -2.0 * (k.kapx + k.kapy);
    k.b2 = 2.0 * (g.beta - 1.0); k.omb2 = 1.0 - k.b2;
    k.j0 = (int)blockIdx.y * rows; k.j1 = min(k.j0 + rows, g.ny);
    k.ylo = max(k.j0 - 2, -1); k.ycnt = g.ny + 1 - k.ylo;
    k.px = g.side[SIDE_XLO].kind == BC_PERIODIC; k.py = g.side[SIDE_YLO].kind == BC_PERIODIC;
    k.any_src = false; k.any_refl = false;
    const long long step_no = clk->steps;
    k.src = src_buffer(g, step_no);
    const int c = tid & (WS_COLS - 1);                             // column of the strip
    const int i = (int)blockIdx.x * (WS_COLS - 6) - 3 + c;         // column on the ghost-extended mesh
    const int r0 = k.j0 - 3, rend = k.j1 + 6;                      // the Y group runs behind, output row = r - 6
    double smx = 0.0, smy = 0.0;
    int flags = 0;
    __syncthreads();                                               // (the fill above is complete)

    if (tid < WS_COLS) {
        // ================================= X group: the x-sweep =======================================================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 96;");
        XThread th;
        th.i = i;
        th.cm = map_column(g, i);
        th.special = (th.cm.neg2 ? 4 : 0) | (th.cm.xsrc >= 0 ? 8 : 0);
        th.p = smem + (c + 1) * 16;
        th.pq = smem + ws_ring_off() + c * 8;
        th.smx = 0.0; th.mqx = th.mdx = 0x7fffffff;
        th.w = {0.0, 1.0, 0.0, 0.0, -1.0, 0.0, 0.0, 0.0};
        th.rn1 = th.rn2 = 0.5;
        th.cx = {1.0, 0.0, 0.0, 0.0, 0.0};
        for (int d = 0; d < 2; ++d) th.aq[d][0] = 1.0, th.aq[d][1] = th.aq[d][2] = 0.0;
        for (int d = 0; d < 2; ++d) {                              // rows r0 and r0+1 start their way into the ring
            const RowMap rm = map_row(g, r0 + d);
            const size_t idx = (size_t)rm.row * g.nx + th.cm.col;
            char* pd = th.pq + ((r0 + d) & 3) * (3 * WS_COLS * 8);
            cp_async8(pd, q1 + idx); cp_async8(pd + WS_COLS * 8, q2 + idx); cp_async8(pd + 2 * WS_COLS * 8, q3 + idx);
            cp_async_commit();
        }
        int t = r0 - 2;                                            // two ticks of pipeline fill before the Y warps start
        const int slo = 0, shi = min(rend - 1, g.ny - 5);          // steady: rows t .. t+4 are interior rows, t >= r0
        while (t < rend && (t < max(slo, r0) || (t & 1))) {
            if (t & 1) ws_xtick<1, false>(g, k, th, t, r0, q1, q2, q3); else ws_xtick<0, false>(g, k, th, t, r0, q1, q2, q3);
            ++t;
        }
        for (; t + 1 <= shi; t += 2) {
            ws_xtick<0, true>(g, k, th, t, r0, q1, q2, q3);
            ws_xtick<1, true>(g, k, th, t + 1, r0, q1, q2, q3);
        }
        while (t < rend) {
            if (t & 1) ws_xtick<1, false>(g, k, th, t, r0, q1, q2, q3); else ws_xtick<0, false>(g, k, th, t, r0, q1, q2, q3);
            ++t;
        }
        cp_async_wait<0>();
        const bool x_if_m = c >= 1 && i >= 0 && i <= g.nx;          // x-interface i-1/2 touches an interior cell
        const bool x_if_f = c >= 1 && i >= -1 && i <= g.nx + 1;     // ... is one the scheme solves
        const bool x_cell = i >= -2 && i <= g.nx + 1;
        if (x_cell && th.mqx <= 0) flags |= F_ENONPOS;
        if (x_if_f && th.mdx < 0) flags |= F_ENONREAL;
        if (x_if_m) smx = th.smx;
    } else {
        // ================================= Y group: the y-sweep and the source step ===================================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 160;");
        YThread th;
        th.i = i;
        th.special = (!k.px && i == 0 ? 1 : 0) | (!k.px && i == g.nx - 1 ? 2 : 0);
        th.out_col = c >= 3 && c <= WS_COLS - 4 && i >= 0 && i < g.nx;
        th.p = smem + (c + 1) * 16;
        th.smy = 0.0; th.mqy = th.mdy = 0x7fffffff; th.mxo = 0;
        YSet Y0, Y1;
        Y0.c = {1.0, 0.0, 0.0, 0.0, 0.0};
        Y0.w = {0.0, 1.0, 0.0, 0.0, -1.0, 0.0, 0.0, 0.0};
        Y0.rn1 = Y0.rn2 = 0.5; Y0.pb1 = Y0.pb2 = Y0.pb3 = 0.0;
        Y1 = Y0;
        YCarry cy;
        cy.gp1 = cy.gp2 = cy.gp3 = cy.gf1 = 0.0;
        cy.q1 = 1.0; cy.q2 = cy.q3 = 0.0;
        cy.c1 = 1.0; cy.c2 = cy.c3 = cy.zC2 = cy.zC3 = cy.zS2 = cy.zS3 = 0.0;
        cy.pend = Y0.c;
        int r = r0;
        // steady: the interface solved (I(ry-1), ry = r-1) is a real one, output row r-6 >= j0 and away from the y edges
        const int slo = max(k.j0 + 6, k.py ? 0 : 7), shi = min(rend - 1, g.ny);
        while (r < rend && (r < slo || (r & 1))) {
            if (r & 1) ws_ytick<1, false>(g, k, th, cy, Y0, Y1, r, o1, o2, o3); else ws_ytick<0, false>(g, k, th, cy, Y0, Y1, r, o1, o2, o3);
            ++r;
        }
        for (; r + 1 <= shi; r += 2) {
            ws_ytick<0, true>(g, k, th, cy, Y0, Y1, r, o1, o2, o3);
            ws_ytick<1, true>(g, k, th, cy, Y0, Y1, r + 1, o1, o2, o3);
        }
        while (r < rend) {
            if (r & 1) ws_ytick<1, false>(g, k, th, cy, Y0, Y1, r, o1, o2, o3); else ws_ytick<0, false>(g, k, th, cy, Y0, Y1, r, o1, o2, o3);
            ++r;
        }
        const bool y_col = c >= 2 && c <= WS_COLS - 3 && i >= 0 && i < g.nx;
        if (y_col && th.mqy <= 0) flags |= F_ENONPOS;
        if (y_col && th.mdy < 0) flags |= F_ENONREAL;
        if (th.mxo >= 0x7ff00000) flags |= F_ENAN;
        if (y_col) smy = th.smy;
    }
    // ---- analytic ghost cells of the NEXT step, t_{n+1} = t_n + dt_n (known since this step began), into the other buffer:
    // every block's Y warps (the larger register budget) take a slice of the records
    if (k.src && more && tid >= WS_COLS) {
        const double t_next = __dadd_rn(k.t, clk->dt);
        double* out = src_buffer(g, step_no + 1);
        const size_t recs = src_off(g.nx, g.ny, 4) / 3, nblk = (size_t)gridDim.x * gridDim.y;
        for (size_t n = ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * WS_COLS + (tid - WS_COLS); n < recs; n += nblk * WS_COLS)
            source_record(g, t_next, n, out);
    }
    // ---- reductions: M of and the sticky flags ---------------------------------------------------------
    __syncthreads();
    block_max_to(&clk->sx_bits, smx);
    __syncthreads();
    block_max_to(&clk->sy_bits, smy);
    block_flags_to(&clk->flags, flags);
    // ---- the block that finishes last ends the step (clock) ----------------------------------------------------------
    step_tail(g, clk, value, mode, more);
}

}  // namespace fvnl
