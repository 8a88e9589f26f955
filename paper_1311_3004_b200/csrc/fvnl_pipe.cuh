// fvnl_pipe.cuh -- the one-pass step kernel with the x-sweep software-pipelined over rows: ONE barrier per tick.
//
// Same mapping and arithmetic as fvnl_fused.cuh (one thread = one column, a block marches over a chunk of rows,
// x-neighbours through shared memory, y-neighbours in registers).  What changes is the schedule.  The x-sweep of a row
// is a chain cell -> Riemann solve -> limited flux -> update with a neighbour exchange between any two links; in
// fvnl_fused.cuh the chain of ONE row runs inside a tick, three barriers apart, and the warp's FP64 dependency
// latency (9 cycles per dependent op, measured) is exposed: the kernel is latency bound at 12 warps per SM.  Here a
// tick t works on FOUR rows at once,
//     cells of row t | Riemann solves of row t-1 | limited fluxes of row t-2 | update (27) of row t-3 -> Q*(., t-3)
// plus the y-sweep on Q*(., t-4) and the source step (output row t-7): six independent instruction streams in one
// basic block.  Everything a stream reads from other threads was published in the previous tick, everything it
// publishes goes to the other half of a double-buffered shared-memory record, so one barrier per tick suffices.
#pragma once
#include "fvnl_fused.cuh"

namespace fvnl {

// Shared memory: the ten double2 arrays of fvnl_fused.cuh, each twice (tick parity), then an 8-slot prefetch ring.
template <int BX> __host__ __device__ constexpr int pp_off(int k, int parity) { return (2 * k + parity) * (BX + 2) * 16; }
template <int BX> __host__ __device__ constexpr int pipe_ring_off() { return pp_off<BX>(SM_ARRAYS, 0); }
template <int BX> __host__ __device__ constexpr int pipe_smem_bytes() { return pipe_ring_off<BX>() + 8 * pre_slot_bytes<BX>(); }

// Rolling x-state of the rows of one parity: the cell of row rho (written at tick rho), the waves of its interface
// i-1/2 (tick rho+1), the right-going part of that interface (tick rho+2; consumed at tick rho+3).
struct XSet {
    Cx c;
    Wv w;
    double rn1, rn2;
    double p1, p2, p3;
};

struct PipeCarry {
    double s1, s2, s3;                       // Q*(., t-4) for the y-sweep (left by the previous tick)
    double gp1, gp2, gp3;                    // right-going part of the y-interface below the newest one, y-form
    double c1, c2, c3, zC2, zC3;             // Q**(ry-3) and its z
    double zS2, zS3;                         // z of Q**(ry-4)
};

// One tick.  P = t & 1 (compile time): this tick publishes into the shared-memory arrays of parity P and reads what
// the previous tick published (parity P^1).  X[P] holds rows t, t-2; X[P^1] rows t-1, t-3.  Y[P] becomes the set of
// the newest y-interface (ry-1/2, ry = t-4), Y[P^1] is the one below it.  STEADY as in fvnl_fused.cuh.
template <int BX, int P, bool STEADY>
__device__ __forceinline__ void ptick(const Grid& g, const StepK& k, ThreadK& th, PipeCarry& cy, XSet& X0, XSet& X1,
                                      YSet& Y0, YSet& Y1, int t, const double* __restrict__ q1,
                                      const double* __restrict__ q2, const double* __restrict__ q3,
                                      double* __restrict__ o1, double* __restrict__ o2, double* __restrict__ o3) {
    XSet& XP = P ? X1 : X0;
    XSet& XQ = P ? X0 : X1;
    YSet& N = P ? Y1 : Y0;
    const YSet& A = P ? Y0 : Y1;
    constexpr int W = P, R = P ^ 1;                                           // parities written / read
    char* const p = th.p;
    const int ry = t - 4;
    RowMap rm, rm_pre;                                                        // rows t and t+2 (the one to prefetch)
    if (STEADY) {
        rm.row = t; rm.neg3 = false; rm.ysrc = -1;
        rm_pre.row = t + 2;
    } else {
        rm = map_row(g, t);
        rm_pre = map_row(g, t + 2);
    }
    // ---- cells of row t (prefetch row t+2) -----------------------------------------------------------------------
    cp_async_wait<1>();                                                       // row t has landed
    double a1, a2, a3;
    {
        char* ps = th.pq + (t & 7) * pre_slot_bytes<BX>();
        a1 = lds1(ps); a2 = lds1(ps + BX * 8); a3 = lds1(ps + 2 * BX * 8);
        char* pd = th.pq + ((t + 2) & 7) * pre_slot_bytes<BX>();
        const size_t idx = (size_t)rm_pre.row * g.nx + th.cm.col;
        cp_async8(pd, q1 + idx); cp_async8(pd + BX * 8, q2 + idx); cp_async8(pd + 2 * BX * 8, q3 + idx);
        cp_async_commit();
        if ((th.special & 12) || (!STEADY && (rm.neg3 || rm.ysrc >= 0))) {    // ghost column / row with a rule: rare
            if (!STEADY && rm.neg3) a3 = -a3;
            if (th.special & 4) a2 = -a2;
            if ((th.special & 8) || (!STEADY && rm.ysrc >= 0)) {
                const double3 s = apply_sources(g, th.cm.xsrc, rm.ysrc, th.cm.col, th.cm.neg2, th.i, t, k.t, a1, a2, a3);
                a1 = s.x; a2 = s.y; a3 = s.z;
            }
            sts1(ps, a1); sts1(ps + BX * 8, a2); sts1(ps + 2 * BX * 8, a3);   // the update of row t reads them back
        }
    }
    // Each of the three steps below is evaluated as a PAIR (fvnl_pair.cuh): lane a = the x-sweep's problem, lane b = the
    // y-sweep's, so that two independent instructions sit next to each other along every dependency chain.
    const double b1o = N.c.q1, b2o = N.c.q2, b3o = N.c.q3;                    // Q*(ry-2), y-form (before N is overwritten)
    I2 tq2 = {0x7fffffff, 0x7fffffff}, td2 = tq2;
    {   // cells: row t of Q^n | Q*(., ry) with positions 2,3 switched
        const CxT<V2> c2 = cell_of(pk(a1, cy.s1), pk(a2, cy.s3), pk(a3, cy.s2), tq2);
        XP.c = lane_a(c2);
        N.c = lane_b(c2);
    }
    sts2(p + pp_off<BX>(0, W), XP.c.q1, XP.c.q2); sts2(p + pp_off<BX>(1, W), XP.c.q3, XP.c.hz2);
    sts1(p + pp_off<BX>(2, W), XP.c.hz3);

    WvT<V2> w2;                                                               // row t-1 at i-1/2 | column at ry-1/2
    V2 rn1, rn2;
    {   // Riemann solves: x-interface i-1/2 of row t-1 (its cells were published last tick) | y-interface ry-1/2
        Cx L;
        const double2 u0 = lds2(p + pp_off<BX>(0, R) - 16), u1 = lds2(p + pp_off<BX>(1, R) - 16);
        L.q1 = u0.x; L.q2 = u0.y; L.q3 = u1.x; L.hz2 = u1.y; L.hz3 = lds1(p + pp_off<BX>(2, R) - 16);
        w2 = riemann2(pk(L, A.c), pk(XQ.c, N.c), k.b2, k.omb2, td2);
        rn1 = rnorm(w2.s1, w2.r31); rn2 = rnorm(w2.s2, w2.r32);
        XQ.w = lane_a(w2); XQ.rn1 = rn1.a; XQ.rn2 = rn2.a;
        N.w = lane_b(w2); N.rn1 = rn1.b; N.rn2 = rn2.b;
        sts2(p + pp_off<BX>(3, W), XQ.w.al1, XQ.w.s1); sts2(p + pp_off<BX>(4, W), XQ.w.r31, XQ.w.al3);
        sts2(p + pp_off<BX>(5, W), XQ.w.al2, XQ.w.s2); sts1(p + pp_off<BX>(6, W), XQ.w.r32);
    }

    Fl G;
    {   // limited fluxes: x-interface of row t-2 (its waves were published last tick) | y-interface ry-3/2 (A)
        const Wv& w = XP.w;
        const char* u1 = p + (hi_word(w.s1) < 0 ? 16 : -16);                  // upwind interface
        const char* u2 = p + (hi_word(w.s2) < 0 ? 16 : -16);
        const char* u3 = p + (hi_word(w.v) < 0 ? 16 : -16);
        const double2 k1 = lds2(u1 + pp_off<BX>(3, R)), k2 = lds2(u2 + pp_off<BX>(5, R));
        const double k1r = lds1(u1 + pp_off<BX>(4, R)), k2r = lds1(u2 + pp_off<BX>(6, R)), k3 = lds1(u3 + pp_off<BX>(4, R) + 8);
        // r_K.r_k: x with the upwind neighbour's waves | y between A and N (symmetric: serves both of them)
        const V2 d1 = rdot(pk(k1.y, A.w.s1), pk(k1r, A.w.r31), pk(w.s1, N.w.s1), pk(w.r31, N.w.r31));
        const V2 d2 = rdot(pk(k2.y, A.w.s2), pk(k2r, A.w.r32), pk(w.s2, N.w.s2), pk(w.r32, N.w.r32));
        const V2 c1 = pk(k1.x, N.w.al1) * d1 * pk(XP.rn1, A.rn1);             // x: b1 | y: b1 of A if N is its upwind side
        const V2 c2 = pk(k2.x, N.w.al2) * d2 * pk(XP.rn2, A.rn2);
        N.pb1 = A.w.al1 * d1.b * N.rn1; N.pb2 = A.w.al2 * d2.b * N.rn2; N.pb3 = A.w.al3;   // if A is N's upwind side
        const V2 b1 = pk(c1.a, hi_word(A.w.s1) < 0 ? c1.b : A.pb1);
        const V2 b2 = pk(c2.a, hi_word(A.w.s2) < 0 ? c2.b : A.pb2);
        const V2 b3 = pk(k3, hi_word(A.w.v) < 0 ? N.w.al3 : A.pb3);
        const FlT<V2> F2 = flux2(pk(w, A.w), b1, b2, b3, pk(k.lamx, k.lamy));
        const Fl F = lane_a(F2);
        G = lane_b(F2);
        sts2(p + pp_off<BX>(7, W), F.m1, F.m2); sts1(p + pp_off<BX>(8, W), F.m3);
        XP.p1 = F.p1; XP.p2 = F.p2; XP.p3 = F.p3;
    }
    if (STEADY || (unsigned)t < (unsigned)g.ny) th.mqx = min(th.mqx, tq2.a);
    if (STEADY || (t - 1 >= k.j0 - 3 && (unsigned)(t - 1) < (unsigned)g.ny)) {
        th.mdx = min(th.mdx, td2.a);
        th.smx = dmax(th.smx, fabs(hi_word(XQ.w.v) < 0 ? XQ.w.s2 : XQ.w.s1));       // max(|s1|,|s2|) = |v| + a
    }
    if (STEADY || (unsigned)(ry - k.ylo) <= (unsigned)k.ycnt) {               // y-interface ry-1/2 is one the scheme solves
        th.mqy = min(th.mqy, tq2.b); th.mdy = min(th.mdy, td2.b);
        if (STEADY || (unsigned)ry <= (unsigned)g.ny) th.smy = dmax(th.smy, fabs(hi_word(N.w.v) < 0 ? N.w.s2 : N.w.s1));
    }

    // ---- update (27) of row t-3 -> Q*(., t-3), handed to the y-sweep of the next tick ---------------------------------
    double sn1, sn2, sn3;
    {
        const double2 gm = lds2(p + pp_off<BX>(7, R) + 16);
        const double gm3 = lds1(p + pp_off<BX>(8, R) + 16);
        const char* ps = th.pq + ((t - 3) & 7) * pre_slot_bytes<BX>();
        sn1 = fma(-k.lamx, XQ.p1 + gm.x, lds1(ps));
        sn2 = fma(-k.lamx, XQ.p2 + gm.y, lds1(ps + BX * 8));
        sn3 = fma(-k.lamx, XQ.p3 + gm3, lds1(ps + 2 * BX * 8));
    }

    // ---- y-update: Q**(., ry-2) -------------------------------------------------------------------------------------
    const double n1 = fma(-k.lamy, cy.gp1 + G.m1, b1o);                       // physical order n1, n2, n3
    const double n3 = fma(-k.lamy, cy.gp2 + G.m2, b2o);
    const double n2 = fma(-k.lamy, cy.gp3 + G.m3, b3o);
    cy.gp1 = G.p1; cy.gp2 = G.p2; cy.gp3 = G.p3;
    cy.s1 = sn1; cy.s2 = sn2; cy.s3 = sn3;

    // ---- source step (26): x part of row ry-3 (its z was published last tick), publish z of row ry-2, finish ry-3 -----
    double2 zW = lds2(p + pp_off<BX>(9, R) - 16), zE = lds2(p + pp_off<BX>(9, R) + 16);
    if (th.special & 3) {
        if (th.special & 1) zW = ghost_z(g, SIDE_XLO, (ry - 3 + 0.5) * g.dy, -0.5 * g.dx, k.t, cy.zC2, cy.zC3);
        if (th.special & 2) zE = ghost_z(g, SIDE_XHI, (ry - 3 + 0.5) * g.dy, (g.nx + 0.5) * g.dx, k.t, cy.zC2, cy.zC3);
    }
    const double H2 = fma(k.k2, cy.zC2, fma(k.kapx, zE.x + zW.x, cy.c2));
    const double H3 = fma(k.k2, cy.zC3, fma(k.kapx, zE.y + zW.y, cy.c3));
    const double rq = rcp_o1(n1);
    const double zN2 = n2 * rq, zN3 = n3 * rq;
    sts2(p + pp_off<BX>(9, W), zN2, zN3);
    const int Ro = ry - 3;
    if (STEADY || Ro >= k.j0) {                                               // Ro < j1 by the loop bound
        double y2 = zN2 + cy.zS2, y3 = zN3 + cy.zS3;
        if (!STEADY && !k.py && (Ro == 0 || Ro == g.ny - 1)) {
            const double x = (th.i + 0.5) * g.dx;
            double2 lo = make_double2(cy.zS2, cy.zS3), hi = make_double2(zN2, zN3);
            if (Ro == 0) lo = ghost_z(g, SIDE_YLO, x, x, k.t, cy.zC2, cy.zC3);
            if (Ro == g.ny - 1) hi = ghost_z(g, SIDE_YHI, x, x, k.t, cy.zC2, cy.zC3);
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
    __syncthreads();                                                          // the one barrier: parity W is published
}

// The step kernel.  grid = (strips, chunks); block = BX threads; dynamic shared memory = pipe_smem_bytes<BX>().
template <int BX, int MINB>
__global__ void __launch_bounds__(BX) __maxnreg__((65536 / (BX * MINB)) / 8 * 8 > 255 ? 255 : (65536 / (BX * MINB)) / 8 * 8)
k_step_pipe(Grid g, Clock* clk, const double* __restrict__ q1, const double* __restrict__ q2,
            const double* __restrict__ q3, double* __restrict__ o1, double* __restrict__ o2, double* __restrict__ o3,
            int rows) {
    extern __shared__ __align__(16) char smem[];
    const int tid = threadIdx.x;
    for (int j = tid; j < pipe_smem_bytes<BX>() / 8; j += BX) reinterpret_cast<double*>(smem)[j] = 1.0;   // finite fill

    StepK k;
    k.t = clk->t; k.lamx = clk->lamx; k.lamy = clk->lamy; k.kapx = clk->kapx; k.kapy = clk->kapy;
    k.k2 = -2.0 * (k.kapx + k.kapy);
    k.b2 = 2.0 * (g.beta - 1.0); k.omb2 = 1.0 - k.b2;
    k.j0 = (int)blockIdx.y * rows; k.j1 = min(k.j0 + rows, g.ny);
    k.ylo = max(k.j0 - 2, -1); k.ycnt = g.ny + 1 - k.ylo;
    k.px = g.side[SIDE_XLO].kind == BC_PERIODIC; k.py = g.side[SIDE_YLO].kind == BC_PERIODIC;
    k.any_src = false; k.any_refl = false;

    ThreadK th;
    th.i = (int)blockIdx.x * (BX - 6) - 3 + tid;
    th.cm = map_column(g, th.i);
    th.special = (!k.px && th.i == 0 ? 1 : 0) | (!k.px && th.i == g.nx - 1 ? 2 : 0) | (th.cm.neg2 ? 4 : 0) |
                 (th.cm.xsrc >= 0 ? 8 : 0);
    th.out_col = tid >= 3 && tid <= BX - 4 && th.i >= 0 && th.i < g.nx;
    th.p = smem + (tid + 1) * 16;
    th.pq = smem + pipe_ring_off<BX>() + tid * 8;
    th.smx = 0.0; th.smy = 0.0;
    th.mqx = th.mdx = th.mqy = th.mdy = 0x7fffffff; th.mxo = 0;

    YSet Y0, Y1;
    Y0.c = {1.0, 0.0, 0.0, 0.0, 0.0};
    Y0.w = {0.0, 1.0, 0.0, 0.0, -1.0, 0.0, 0.0, 0.0};
    Y0.rn1 = Y0.rn2 = 0.5; Y0.pb1 = Y0.pb2 = Y0.pb3 = 0.0;
    Y1 = Y0;
    XSet X0, X1;
    X0.c = Y0.c; X0.w = Y0.w; X0.rn1 = X0.rn2 = 0.5; X0.p1 = X0.p2 = X0.p3 = 0.0;
    X1 = X0;
    PipeCarry cy;
    cy.gp1 = cy.gp2 = cy.gp3 = 0.0;
    cy.s1 = 1.0; cy.s2 = cy.s3 = 0.0;
    cy.c1 = 1.0; cy.c2 = cy.c3 = cy.zC2 = cy.zC3 = cy.zS2 = cy.zS3 = 0.0;

    int t = k.j0 - 3;
    const int tend = k.j1 + 7;                                     // output row = t - 7
    __syncthreads();                                               // (the fill above is complete)
    for (int d = 0; d < 2; ++d) {                                  // rows t and t+1 start their way into the ring
        const RowMap rm = map_row(g, t + d);
        const size_t idx = (size_t)rm.row * g.nx + th.cm.col;
        char* pd = th.pq + ((t + d) & 7) * pre_slot_bytes<BX>();
        cp_async8(pd, q1 + idx); cp_async8(pd + BX * 8, q2 + idx); cp_async8(pd + 2 * BX * 8, q3 + idx);
        cp_async_commit();
    }
    // steady ticks t in [slo, shi]: rows t .. t+2 interior, every stage holds real data, output row t-7 >= j0 and
    // away from the y edges
    const int slo = max(k.j0 + 7, k.py ? 0 : 8), shi = min(tend - 1, g.ny - 3);
    while (t < tend && (t < slo || (t & 1))) {                     // pipeline fill (and everything, near the y edges)
        if (t & 1) ptick<BX, 1, false>(g, k, th, cy, X0, X1, Y0, Y1, t, q1, q2, q3, o1, o2, o3);
        else ptick<BX, 0, false>(g, k, th, cy, X0, X1, Y0, Y1, t, q1, q2, q3, o1, o2, o3);
        ++t;
    }
    for (; t + 1 <= shi; t += 2) {
        ptick<BX, 0, true>(g, k, th, cy, X0, X1, Y0, Y1, t, q1, q2, q3, o1, o2, o3);
        ptick<BX, 1, true>(g, k, th, cy, X0, X1, Y0, Y1, t + 1, q1, q2, q3, o1, o2, o3);
    }
    while (t < tend) {
        if (t & 1) ptick<BX, 1, false>(g, k, th, cy, X0, X1, Y0, Y1, t, q1, q2, q3, o1, o2, o3);
        else ptick<BX, 0, false>(g, k, th, cy, X0, X1, Y0, Y1, t, q1, q2, q3, o1, o2, o3);
        ++t;
    }
    cp_async_wait<0>();

    // ---- reductions: M of and the sticky flags, masked by which results of this thread are real ----
    const int i = th.i;
    const bool x_if_m = tid >= 1 && i >= 0 && i <= g.nx;            // x-interface i-1/2 touches an interior cell
    const bool x_if_f = tid >= 1 && i >= -1 && i <= g.nx + 1;       // ... is one the scheme solves
    const bool x_cell = i >= -2 && i <= g.nx + 1;
    const bool y_col = tid >= 2 && tid <= BX - 3 && i >= 0 && i < g.nx;
    int flags = 0;
    if ((x_cell && th.mqx <= 0) || (y_col && th.mqy <= 0)) flags |= F_ENONPOS;
    if ((x_if_f && th.mdx < 0) || (y_col && th.mdy < 0)) flags |= F_ENONREAL;
    if (th.mxo >= 0x7ff00000) flags |= F_ENAN;
    block_max_to(&clk->sx_bits, x_if_m ? th.smx : 0.0);
    __syncthreads();
    block_max_to(&clk->sy_bits, y_col ? th.smy : 0.0);
    block_flags_to(&clk->flags, flags);
}

}  // namespace fvnl
