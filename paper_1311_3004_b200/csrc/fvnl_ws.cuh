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
// (T = double or float: elements of T2, i.e. 16 or 8 bytes)
constexpr int WS_ARRAYS = 12;
template <class T> __host__ __device__ constexpr int ws_elem() { return 2 * (int)sizeof(T); }
template <class T> __host__ __device__ constexpr int ws_arr2(int k, int parity) { return (2 * k + parity) * (WS_COLS + 2) * ws_elem<T>(); }
template <class T> __host__ __device__ constexpr int ws_ring_off() { return 2 * WS_ARRAYS * (WS_COLS + 2) * ws_elem<T>(); }
template <class T> __host__ __device__ constexpr int ws_slot() { return 3 * WS_COLS * (int)sizeof(T); }       // one row of the prefetch ring
template <class T> __host__ __device__ constexpr int ws_smem_bytes() { return ws_ring_off<T>() + 4 * ws_slot<T>(); }

__device__ __forceinline__ void bar_x() { asm volatile("bar.sync 1, 128;" ::: "memory"); }
__device__ __forceinline__ void bar_all() { asm volatile("bar.sync 2, 256;" ::: "memory"); }

template <class T> struct XThreadT {
    ColMap cm;
    int i, special;
    char *p, *pq;
    T smx;
    int mqx, mdx;
    WvT<T> w;                                // waves of interface i-1/2 of the row solved in the previous tick
    T rn1, rn2;                              // and their 1/(r.r)
    CxT<T> cx;                               // this column's cell of the row converted in the previous tick
    T aq[2][3];                              // Q^n(i, .) of the rows loaded in the previous two ticks, by row parity
    const double* srow;                      // ghost column of a SOURCE x-side: its records of this step (record of row r at
    double s1, s2, s3;                       // srow + 3 r), and the record of the row phase A converts NEXT, loaded one tick
};                                           // ahead (an L2 round trip inside the tick stalls the whole warp)

// The analytic record of row r for a ghost column of a SOURCE x-side (q1 <= 0: none / outside the aperture).
template <class T> __device__ __forceinline__ void x_prefetch_source(const Grid& g, XThreadT<T>& th, int r) {
    if (th.srow && r >= -3 && r <= g.ny + 2) { const double* sp = th.srow + 3 * r; th.s1 = sp[0]; th.s2 = sp[1]; th.s3 = sp[2]; }
    else th.s1 = -1.0;
}

// Density variable of a cell from a full-form fp64 value (analytic ghost cells): q1, or rho' = q1 - 1 in fp32.
template <class T> __device__ __forceinline__ T dens_var(double q1) { return Num<T>::perturbation ? T(q1 - 1.0) : T(q1); }

// One tick of an X warp.  The x-sweep is software-pipelined over rows: tick t runs three INDEPENDENT pieces of work, each on
// its own row, so that the warp has several dependency chains to issue from (a dependent FP64 operation waits 9 cycles) and
// ONE block-wide barrier per tick separates everything:
//   phase C, row t   : limited fluxes (28)-(30) of interface i-1/2 from its waves (solved in tick t-1, kept in registers)
//                      and the upwind neighbour's (shared memory) -> the two halves of the update (27) for the Y warps;
//   phase B, row t+1 : Riemann solve between the cells of columns i-1 and i (converted in tick t-1)
//                      -> waves to shared memory;
//   phase A, row t+2 : Q^n(., t+2) from the prefetch ring, ghost rule, primitive conversion -> cell to shared memory;
//                      prefetch of row t+4.
// P = t & 1.  The two ticks before r0 are pipeline fill: the Y warps are not running yet and the barrier is the X group's own.
template <class T, int P, bool STEADY>
__device__ __forceinline__ void ws_xtick(const Grid& g, const StepKT<T>& k, XThreadT<T>& th, int t, int r0,
                                         const T* __restrict__ q1, const T* __restrict__ q2, const T* __restrict__ q3) {
    char* const p = th.p;
    constexpr int Q = P ^ 1;
    constexpr int E = ws_elem<T>();                                           // bytes from one column's element to the next
    constexpr int S = (int)sizeof(T);
    // ---- phase C: row t ----------------------------------------------------------------------------------------------
    if (STEADY || t >= r0) {
        const WvT<T>& w = th.w;
        const char* u1 = p + (Num<T>::hi(w.s1) < 0 ? E : -E);                 // upwind interface
        const char* u2 = p + (Num<T>::hi(w.s2) < 0 ? E : -E);
        const char* u3 = p + (Num<T>::hi(w.v) < 0 ? E : -E);
        const auto k1 = ldp<T>(u1 + ws_arr2<T>(3, P)), k2 = ldp<T>(u2 + ws_arr2<T>(5, P));
        const T k1r = ld1<T>(u1 + ws_arr2<T>(4, P)), k2r = ld1<T>(u2 + ws_arr2<T>(6, P)), k3 = ld1<T>(u3 + ws_arr2<T>(4, P) + S);
        const T own1 = th.aq[P][0], own2 = th.aq[P][1], a3 = th.aq[P][2];     // Q^n(i, t), loaded two ticks ago
        const T b1 = k1.x * rdot(k1.y, k1r, w.s1, w.r31) * th.rn1;
        const T b2 = k2.x * rdot(k2.y, k2r, w.s2, w.r32) * th.rn2;
        const FlT<T> F = flux2(w, b1, b2, k3, k.lamx);
        // the two halves of (27) for row t: what this interface sends left, and this column's own part
        // (the density component goes over unrounded: q1, p1 and the first component of F~, see update_q1)
        sts2(p + ws_arr2<T>(7, P), F.m1, F.m2); sts2(p + ws_arr2<T>(8, P), F.m3, F.ft1);
        sts2(p + ws_arr2<T>(9, P), own1, fma(-k.lamx, F.p2, own2));
        sts2(p + ws_arr2<T>(10, P), fma(-k.lamx, F.p3, a3), F.p1);
    }
    // ---- phase B: row t+1 --------------------------------------------------------------------------------------------
    if (STEADY || t + 1 >= r0) {
        CxT<T> L;
        const CxT<T> C = th.cx;
        {
            const auto l0 = ldp<T>(p + ws_arr2<T>(0, Q) - E), l1 = ldp<T>(p + ws_arr2<T>(1, Q) - E);
            L.q1 = l0.x; L.q2 = l0.y; L.q3 = l1.x; L.hz2 = l1.y; L.hz3 = ld1<T>(p + ws_arr2<T>(2, Q) - E);
        }
        int td = 0x7fffffff;
        const WvT<T> w = riemann2(L, C, k.b2, k.omb2, td);
        th.rn1 = rnorm(w.s1, w.r31); th.rn2 = rnorm(w.s2, w.r32);
        th.w = w;
        sts2(p + ws_arr2<T>(3, Q), w.al1, w.s1); sts2(p + ws_arr2<T>(4, Q), w.r31, w.al3); sts2(p + ws_arr2<T>(5, Q), w.al2, w.s2);
        sts1(p + ws_arr2<T>(6, Q), w.r32);
        if (STEADY || (unsigned)(t + 1) < (unsigned)g.ny) {
            th.mdx = min(th.mdx, td);
            th.smx = Num<T>::max2(th.smx, fabs(Num<T>::hi(w.v) < 0 ? w.s2 : w.s1));   // max(|s1|,|s2|) = |v| + a
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
        T a1, a2, a3;
        {
            const char* ps = th.pq + (r & 3) * ws_slot<T>();
            a1 = ld1<T>(ps); a2 = ld1<T>(ps + WS_COLS * S); a3 = ld1<T>(ps + 2 * WS_COLS * S);
            char* pd = th.pq + ((r + 2) & 3) * ws_slot<T>();
            const size_t idx = (size_t)rm_pre.row * g.nx + th.cm.col;
            cp_async_elem(pd, q1 + idx); cp_async_elem(pd + WS_COLS * S, q2 + idx); cp_async_elem(pd + 2 * WS_COLS * S, q3 + idx);
            cp_async_commit();
        }
        if ((th.special & 12) || (!STEADY && (rm.neg3 || rm.ysrc >= 0))) {    // ghost column / row with a rule: rare
            if (!STEADY && rm.neg3) a3 = -a3;
            if (th.special & 4) a2 = -a2;
            bool done = false;                                                // x rule first, then y rule (as load_mapped)
            if (th.special & 8) {                                             // record loaded in the previous tick
                if (th.s1 > 0.0) { a1 = dens_var<T>(th.s1); a2 = T(th.s2); a3 = T(th.s3); done = true; }
                x_prefetch_source(g, th, r + 1);
            }
            if (!STEADY && !done && rm.ysrc >= 0) {
                const int sd = rm.ysrc, l = sd == SIDE_YLO ? -1 - r : r - g.ny;
                if (l < 3) {
                    const double* sp = k.src + src_off(g.nx, g.ny, sd) + 3 * ((size_t)g.nx * l + th.cm.col);
                    if (sp[0] > 0.0) { a1 = dens_var<T>(sp[0]); a2 = T(th.cm.neg2 ? -sp[1] : sp[1]); a3 = T(sp[2]); }
                }
            }
        }
        int tq = 0x7fffffff;
        const CxT<T> cx = cell_of(a1, a2, a3, tq);
        sts2(p + ws_arr2<T>(0, P), cx.q1, cx.q2); sts2(p + ws_arr2<T>(1, P), cx.q3, cx.hz2); sts1(p + ws_arr2<T>(2, P), cx.hz3);
        th.cx = cx;
        th.aq[P][0] = a1; th.aq[P][1] = a2; th.aq[P][2] = a3;
        if (STEADY || (unsigned)r < (unsigned)g.ny) th.mqx = min(th.mqx, tq);
    }
    if (!STEADY && t < r0) bar_x(); else bar_all();                           // the Y warps join at tick r0
}

// z of the one-deep ghost of Q** at a non-periodic edge, from the z of the interior cell next to it (reading A9): EXTRAP
// copies, REFLECT negates the normal velocity, SOURCE takes the analytic cell of layer 0 (record `m`: the row for an x
// side, the column for a y side) if it lies inside the aperture.
template <class T>
__device__ __forceinline__ typename Num<T>::T2 ghost_z_plain(const Grid& g, const double* __restrict__ src, int sd, int m, T z2, T z3) {
    const int kind = g.side[sd].kind;
    if (kind == BC_REFLECT) return sd < 2 ? Num<T>::make2(-z2, z3) : Num<T>::make2(z2, -z3);
    if (kind == BC_SOURCE) {
        m = sd < 2 ? min(max(m, -3), g.ny + 2) : min(max(m, 0), g.nx - 1);          // (halo threads / pipeline fill: value unused)
        const double* sp = src + src_off(g.nx, g.ny, sd) + 3 * (size_t)(sd < 2 ? m + 3 : m);
        if (sp[0] > 0.0) {
            const double rc = rcp_o1(sp[0]);
            return Num<T>::make2(T(sp[1] * rc), T(sp[2] * rc));
        }
    }
    return Num<T>::make2(z2, z3);
}

template <class T> struct YThreadT {
    int i, special;
    bool out_col;
    char* p;
    T smy;
    int mqy, mdy, mxo;
    const double* grow;                      // edge column next to a SOURCE x-side: layer-0 records of that side (row m at
    double g1, g2, g3;                       // grow + 3 m), and the record the NEXT tick's source step needs, loaded ahead
};

template <class T> __device__ __forceinline__ void y_prefetch_source(const Grid& g, YThreadT<T>& th, int m) {
    if (th.grow) { m = min(max(m, -3), g.ny + 2); const double* sp = th.grow + 3 * m; th.g1 = sp[0]; th.g2 = sp[1]; th.g3 = sp[2]; }
}

// z of the one-deep ghost of Q** at an x edge from the record loaded ahead (y_prefetch_source), else by the plain rule.
template <class T>
__device__ __forceinline__ typename Num<T>::T2 ghost_z_x(const Grid& g, const YThreadT<T>& th, int sd, T z2, T z3) {
    const int kind = g.side[sd].kind;
    if (kind == BC_REFLECT) return Num<T>::make2(-z2, z3);
    if (kind == BC_SOURCE && th.g1 > 0.0) {
        const double rc = rcp_o1(th.g1);
        return Num<T>::make2(T(th.g2 * rc), T(th.g3 * rc));
    }
    return Num<T>::make2(z2, z3);
}

template <class T> struct YCarryT {
    T gp1, gp2, gp3, gf1;                    // right-going part (and F~, comp. 1) of the y-interface below B
    T q1, q2, q3;                            // Q*(., ry-4), y-form
    T c1, c2, c3, zC2, zC3;                  // Q**(ry-5) and its z
    T zS2, zS3;                              // z of Q**(ry-6)
    CxT<T> pend;                             // cell of Q*(., ry-1), y-form: converted in the previous tick, solved in this one
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
template <class T, int P, bool STEADY>
__device__ __forceinline__ void ws_ytick(const Grid& g, const StepKT<T>& k, YThreadT<T>& th, YCarryT<T>& cy, YSetT<T>& Y0,
                                         YSetT<T>& Y1, int r, T* __restrict__ o1, T* __restrict__ o2, T* __restrict__ o3) {
    YSetT<T>& N = P ? Y1 : Y0;
    YSetT<T>& A = P ? Y0 : Y1;
    constexpr int R = P ^ 1;
    constexpr int E = ws_elem<T>();
    constexpr int S = (int)sizeof(T);
    char* const p = th.p;
    const int ry = r - 1;
    // ---- chain 2: flux of B, Q**(., ry-4), source step ----------------------------------------------------------------
    const FlT<T> G = flux2(N.w, N.pb1, N.pb2, N.pb3, k.lamy);                 // N still holds B
    const T n1 = update_q1(cy.q1, k.lamy, cy.gp1 + G.m1, cy.gf1, G.ft1);      // Q**(i, ry-4); physical order n1, n2, n3
    const T n3 = fma(-k.lamy, cy.gp2 + G.m2, cy.q2);
    const T n2 = fma(-k.lamy, cy.gp3 + G.m3, cy.q3);
    cy.gp1 = G.p1; cy.gp2 = G.p2; cy.gp3 = G.p3; cy.gf1 = G.ft1;
    cy.q1 = N.c.q1; cy.q2 = N.c.q2; cy.q3 = N.c.q3;                           // Q*(ry-3), y-form: next tick's lower row
    auto zW = ldp<T>(p + ws_arr2<T>(11, R) - E), zE = ldp<T>(p + ws_arr2<T>(11, R) + E);   // z of row ry-5, published last tick
    if (th.special & 3) {                                                     // (record of row ry-5 loaded in the previous tick)
        if (th.special & 1) zW = ghost_z_x<T>(g, th, SIDE_XLO, cy.zC2, cy.zC3);
        if (th.special & 2) zE = ghost_z_x<T>(g, th, SIDE_XHI, cy.zC2, cy.zC3);
        y_prefetch_source(g, th, ry - 4);
    }
    const T H2 = fma(k.k2, cy.zC2, fma(k.kapx, zE.x + zW.x, cy.c2));
    const T H3 = fma(k.k2, cy.zC3, fma(k.kapx, zE.y + zW.y, cy.c3));
    const T rq = Num<T>::rcp(Num<T>::perturbation ? T(1) + n1 : n1);
    const T zN2 = n2 * rq, zN3 = n3 * rq;
    sts2(p + ws_arr2<T>(11, P), zN2, zN3);
    const int Ro = ry - 5;
    if (STEADY || Ro >= k.j0) {                                               // Ro < j1 by the loop bound
        T y2 = zN2 + cy.zS2, y3 = zN3 + cy.zS3;
        if (!STEADY && !k.py && (Ro == 0 || Ro == g.ny - 1)) {
            auto lo = Num<T>::make2(cy.zS2, cy.zS3), hi = Num<T>::make2(zN2, zN3);
            if (Ro == 0) lo = ghost_z_plain<T>(g, k.src, SIDE_YLO, th.i, cy.zC2, cy.zC3);
            if (Ro == g.ny - 1) hi = ghost_z_plain<T>(g, k.src, SIDE_YHI, th.i, cy.zC2, cy.zC3);
            y2 = hi.x + lo.x; y3 = hi.y + lo.y;
        }
        const T w2 = fma(k.kapy, y2, H2), w3 = fma(k.kapy, y3, H3);
        if (th.out_col) {
            const size_t o = (size_t)Ro * g.nx + th.i;
            o1[o] = cy.c1; o2[o] = w2; o3[o] = w3;
            th.mxo = max(th.mxo, max(Num<T>::hi(cy.c1) & 0x7fffffff, max(Num<T>::hi(w2) & 0x7fffffff, Num<T>::hi(w3) & 0x7fffffff)));
        }
    }
    cy.zS2 = cy.zC2; cy.zS3 = cy.zC3;
    cy.c1 = n1; cy.c2 = n2; cy.c3 = n3; cy.zC2 = zN2; cy.zC3 = zN3;

    // ---- chain 1b: interface N = I(ry-1) between the cells of Q*(ry-2) (A.c) and Q*(ry-1) (cy.pend); limiter inputs of A ----
    int tdy = 0x7fffffff;
    N.c = cy.pend;
    N.w = riemann2(A.c, N.c, k.b2, k.omb2, tdy);
    N.rn1 = rnorm(N.w.s1, N.w.r31); N.rn2 = rnorm(N.w.s2, N.w.r32);
    const T d1 = rdot(A.w.s1, A.w.r31, N.w.s1, N.w.r31), d2 = rdot(A.w.s2, A.w.r32, N.w.s2, N.w.r32);
    N.pb1 = A.w.al1 * d1 * N.rn1; N.pb2 = A.w.al2 * d2 * N.rn2; N.pb3 = A.w.al3;      // if A is N's upwind side
    const T hb1 = N.w.al1 * d1 * A.rn1, hb2 = N.w.al2 * d2 * A.rn2;                   // if N is A's upwind side
    A.pb1 = Num<T>::hi(A.w.s1) < 0 ? hb1 : A.pb1;                             // A's upwind side is now known
    A.pb2 = Num<T>::hi(A.w.s2) < 0 ? hb2 : A.pb2;
    A.pb3 = Num<T>::hi(A.w.v) < 0 ? N.w.al3 : A.pb3;
    if (STEADY || (unsigned)(ry - 1 - k.ylo) <= (unsigned)k.ycnt) {           // I(ry-1) is an interface the scheme solves
        th.mdy = min(th.mdy, tdy);
        if (STEADY || (unsigned)(ry - 1) <= (unsigned)g.ny)
            th.smy = Num<T>::max2(th.smy, fabs(Num<T>::hi(N.w.v) < 0 ? N.w.s2 : N.w.s1));
    }

    // ---- chain 1a: Q*(., ry), the update (27) completed, and its primitive conversion for the next tick ----------------
    {
        const auto u = ldp<T>(p + ws_arr2<T>(9, R)), gm = ldp<T>(p + ws_arr2<T>(7, R) + E);
        const auto u3 = ldp<T>(p + ws_arr2<T>(10, R)), gm3 = ldp<T>(p + ws_arr2<T>(8, R) + E);
        const T ft_own = ld1<T>(p + ws_arr2<T>(8, R) + S);
        const T s1 = update_q1(u.x, k.lamx, u3.y + gm.x, ft_own, gm3.y);
        const T s2 = fma(-k.lamx, gm.y, u.y), s3 = fma(-k.lamx, gm3.x, u3.x);
        int tqy = 0x7fffffff;
        cy.pend = cell_of(s1, s3, s2, tqy);                                   // positions 2,3 switched
        if (STEADY || (unsigned)(ry - k.ylo) <= (unsigned)k.ycnt) th.mqy = min(th.mqy, tqy);   // a cell the y-sweep uses
    }
    bar_all();
}

// Register budgets of the two groups (setmaxnreg) and blocks per SM they are made for.
template <class T> struct WsBudget;
template <> struct WsBudget<double> { static constexpr int blocks_per_sm = 2; };    // compiled for 128: X 96, Y 160
template <> struct WsBudget<float> { static constexpr int blocks_per_sm = 3; };     // compiled for 80:  X 64, Y 96

// The step kernel.  grid = (strips, chunks); block = 256 threads (warps 0-3: X group, warps 4-7: Y group);
// dynamic shared memory = ws_smem_bytes<T>().  setmaxnreg moves registers from the X warps to the Y warps, whose rolling
// window is the large state.  T = double: the state planes hold q; T = float: (rho' = q1 - 1, q2, q3).
// value / mode / more: see step_tail.
template <class T>
__global__ void __launch_bounds__(256, WsBudget<T>::blocks_per_sm)
k_step_ws(Grid g, Clock* clk, const T* __restrict__ q1, const T* __restrict__ q2, const T* __restrict__ q3,
          T* __restrict__ o1, T* __restrict__ o2, T* __restrict__ o3, int rows, double value, int mode, int more) {
    extern __shared__ __align__(16) char smem[];
    const int tid = threadIdx.x;
    // Programmatic dependent launch: let the NEXT step's grid be scheduled as this one's blocks retire, and do everything that
    // needs no global memory (this fill) before waiting for the previous step's grid to complete and flush (its state, the clock).
    asm volatile("griddepcontrol.launch_dependents;");
    for (int j = tid; j < ws_smem_bytes<T>() / (int)sizeof(T); j += 256) reinterpret_cast<T*>(smem)[j] = T(1);   // finite fill
    asm volatile("griddepcontrol.wait;" ::: "memory");

    StepKT<T> k;
    k.t = clk->t; k.lamx = T(clk->lamx); k.lamy = T(clk->lamy); k.kapx = T(clk->kapx); k.kapy = T(clk->kapy);
    k.k2 = T(-2.0 * (clk->kapx + clk->kapy));
    k.b2 = T(2.0 * (g.beta - 1.0)); k.omb2 = T(1.0 - 2.0 * (g.beta - 1.0));
    k.j0 = (int)blockIdx.y * rows; k.j1 = min(k.j0 + rows, g.ny);
    k.ylo = max(k.j0 - 2, -1); k.ycnt = g.ny + 1 - k.ylo;
    k.px = g.side[SIDE_XLO].kind == BC_PERIODIC; k.py = g.side[SIDE_YLO].kind == BC_PERIODIC;
    k.any_src = false; k.any_refl = false;
    const long long step_no = clk->steps;
    k.src = src_buffer(g, step_no);
    const int c = tid & (WS_COLS - 1);                             // column of the strip
    const int i = (int)blockIdx.x * (WS_COLS - 6) - 3 + c;         // column on the ghost-extended mesh
    const int r0 = k.j0 - 3, rend = k.j1 + 6;                      // the Y group runs behind, output row = r - 6
    const T eq1 = Num<T>::perturbation ? T(0) : T(1);              // density variable at equilibrium
    double smx = 0.0, smy = 0.0;
    int flags = 0;
    __syncthreads();                                               // (the fill above is complete)

    if (tid < WS_COLS) {
        // ================================= X group: the x-sweep =======================================================
        if constexpr (sizeof(T) == 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 96;");
        else asm volatile("setmaxnreg.dec.sync.aligned.u32 64;");
        XThreadT<T> th;
        th.i = i;
        th.cm = map_column(g, i);
        th.special = (th.cm.neg2 ? 4 : 0) | (th.cm.xsrc >= 0 ? 8 : 0);
        th.p = smem + (c + 1) * ws_elem<T>();
        th.pq = smem + ws_ring_off<T>() + c * (int)sizeof(T);
        th.smx = T(0); th.mqx = th.mdx = 0x7fffffff;
        th.w = {T(0), T(1), T(0), T(0), T(-1), T(0), T(0), T(0)};
        th.rn1 = th.rn2 = T(0.5);
        th.cx = {eq1, T(0), T(0), T(0), T(0)};
        for (int d = 0; d < 2; ++d) th.aq[d][0] = eq1, th.aq[d][1] = th.aq[d][2] = T(0);
        th.srow = nullptr;
        if (th.cm.xsrc >= 0) {
            const int l = th.cm.xsrc == SIDE_XLO ? -1 - i : i - g.nx;
            if (l < 3) th.srow = k.src + src_off(g.nx, g.ny, th.cm.xsrc) + 3 * ((size_t)(g.ny + 6) * l + 3);
        }
        x_prefetch_source(g, th, r0);                              // the first row phase A converts
        for (int d = 0; d < 2; ++d) {                              // rows r0 and r0+1 start their way into the ring
            const RowMap rm = map_row(g, r0 + d);
            const size_t idx = (size_t)rm.row * g.nx + th.cm.col;
            char* pd = th.pq + ((r0 + d) & 3) * ws_slot<T>();
            cp_async_elem(pd, q1 + idx); cp_async_elem(pd + WS_COLS * (int)sizeof(T), q2 + idx);
            cp_async_elem(pd + 2 * WS_COLS * (int)sizeof(T), q3 + idx);
            cp_async_commit();
        }
        int t = r0 - 2;                                            // two ticks of pipeline fill before the Y warps start
        const int slo = 0, shi = min(rend - 1, g.ny - 5);          // steady: rows t .. t+4 are interior rows, t >= r0
        while (t < rend && (t < max(slo, r0) || (t & 1))) {
            if (t & 1) ws_xtick<T, 1, false>(g, k, th, t, r0, q1, q2, q3); else ws_xtick<T, 0, false>(g, k, th, t, r0, q1, q2, q3);
            ++t;
        }
        for (; t + 1 <= shi; t += 2) {
            ws_xtick<T, 0, true>(g, k, th, t, r0, q1, q2, q3);
            ws_xtick<T, 1, true>(g, k, th, t + 1, r0, q1, q2, q3);
        }
        while (t < rend) {
            if (t & 1) ws_xtick<T, 1, false>(g, k, th, t, r0, q1, q2, q3); else ws_xtick<T, 0, false>(g, k, th, t, r0, q1, q2, q3);
            ++t;
        }
        cp_async_wait<0>();
        const bool x_if_m = c >= 1 && i >= 0 && i <= g.nx;          // x-interface i-1/2 touches an interior cell
        const bool x_if_f = c >= 1 && i >= -1 && i <= g.nx + 1;     // ... is one the scheme solves
        const bool x_cell = i >= -2 && i <= g.nx + 1;
        if (x_cell && th.mqx <= 0) flags |= F_ENONPOS;
        if (x_if_f && th.mdx < 0) flags |= F_ENONREAL;
        if (x_if_m) smx = (double)th.smx;
    } else {
        // ================================= Y group: the y-sweep and the source step ===================================
        if constexpr (sizeof(T) == 8) asm volatile("setmaxnreg.inc.sync.aligned.u32 160;");
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 96;");
        YThreadT<T> th;
        th.i = i;
        th.special = (!k.px && i == 0 ? 1 : 0) | (!k.px && i == g.nx - 1 ? 2 : 0);
        th.out_col = c >= 3 && c <= WS_COLS - 4 && i >= 0 && i < g.nx;
        th.p = smem + (c + 1) * ws_elem<T>();
        th.smy = T(0); th.mqy = th.mdy = 0x7fffffff; th.mxo = 0;
        th.grow = nullptr; th.g1 = -1.0; th.g2 = th.g3 = 0.0;
        if (th.special & 3) {
            const int sd = (th.special & 1) ? SIDE_XLO : SIDE_XHI;             // (nx >= 4: a column is next to one x edge only)
            if (g.side[sd].kind == BC_SOURCE) th.grow = k.src + src_off(g.nx, g.ny, sd) + 3 * 3;
        }
        y_prefetch_source(g, th, r0 - 1 - 5);                                  // row of the first tick's source step
        YSetT<T> Y0, Y1;
        Y0.c = {eq1, T(0), T(0), T(0), T(0)};
        Y0.w = {T(0), T(1), T(0), T(0), T(-1), T(0), T(0), T(0)};
        Y0.rn1 = Y0.rn2 = T(0.5); Y0.pb1 = Y0.pb2 = Y0.pb3 = T(0);
        Y1 = Y0;
        YCarryT<T> cy;
        cy.gp1 = cy.gp2 = cy.gp3 = cy.gf1 = T(0);
        cy.q1 = eq1; cy.q2 = cy.q3 = T(0);
        cy.c1 = eq1; cy.c2 = cy.c3 = cy.zC2 = cy.zC3 = cy.zS2 = cy.zS3 = T(0);
        cy.pend = Y0.c;
        int r = r0;
        // steady: the interface solved (I(ry-1), ry = r-1) is a real one, output row r-6 >= j0 and away from the y edges
        const int slo = max(k.j0 + 6, k.py ? 0 : 7), shi = min(rend - 1, g.ny);
        while (r < rend && (r < slo || (r & 1))) {
            if (r & 1) ws_ytick<T, 1, false>(g, k, th, cy, Y0, Y1, r, o1, o2, o3); else ws_ytick<T, 0, false>(g, k, th, cy, Y0, Y1, r, o1, o2, o3);
            ++r;
        }
        for (; r + 1 <= shi; r += 2) {
            ws_ytick<T, 0, true>(g, k, th, cy, Y0, Y1, r, o1, o2, o3);
            ws_ytick<T, 1, true>(g, k, th, cy, Y0, Y1, r + 1, o1, o2, o3);
        }
        while (r < rend) {
            if (r & 1) ws_ytick<T, 1, false>(g, k, th, cy, Y0, Y1, r, o1, o2, o3); else ws_ytick<T, 0, false>(g, k, th, cy, Y0, Y1, r, o1, o2, o3);
            ++r;
        }
        const bool y_col = c >= 2 && c <= WS_COLS - 3 && i >= 0 && i < g.nx;
        if (y_col && th.mqy <= 0) flags |= F_ENONPOS;
        if (y_col && th.mdy < 0) flags |= F_ENONREAL;
        if (th.mxo >= Num<T>::inf_hi) flags |= F_ENAN;
        if (y_col) smy = (double)th.smy;
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
