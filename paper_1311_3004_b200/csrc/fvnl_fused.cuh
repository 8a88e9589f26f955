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
// The path is bound by instruction issue and the FP64 pipe, not by HBM, so the code below is
// arranged for instruction count: the tick loop is unrolled by two with the roles of the two register sets
// exchanged (no register moves for the rolling window), the upwind neighbour in x is chosen by address, the upwind
// neighbour in y by keeping one "pending" limiter input per wave, shared memory is laid out for 128-bit accesses.
//
// Ghost cells (readings A9, A10, A14 of DESIGN.md) are evaluated on load: the x rule maps the thread's column once,
// the y rule maps the row of each tick; the one-deep ghosts of Q** that the source step needs are derived from the
// neighbouring interior Q** at the edge columns / rows.
#pragma once
#include "fvnl_unfused.cuh"
#include "fvnl_iface.cuh"

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

// Cell (i, r) of the ghost-extended mesh, cm = map_column(g, i): the x rule first, then the y rule (reading A9: a corner
// is the x-ghost of a y-ghost row); analytic cells of SOURCE sides from the buffer `src` of this step (src_buffer), where
// a record with q1 <= 0 means "outside the aperture: extrapolate".
// T = type of the state planes; the cell is returned in full fp64 form (fp32 planes hold rho' = q1 - 1).
template <class T>
__device__ __forceinline__ Q3 load_mapped(const Grid& g, const double* __restrict__ src, const ColMap& cm, int i, int r,
                                          const T* __restrict__ q1, const T* __restrict__ q2, const T* __restrict__ q3) {
    const RowMap rm = map_row(g, r);
    const size_t idx = (size_t)rm.row * g.nx + cm.col;
    Q3 c;
    c.q1 = Num<T>::perturbation ? 1.0 + (double)q1[idx] : (double)q1[idx];
    c.q2 = cm.neg2 ? -(double)q2[idx] : (double)q2[idx];
    c.q3 = rm.neg3 ? -(double)q3[idx] : (double)q3[idx];
    if (cm.xsrc >= 0 && r >= -3 && r <= g.ny + 2) {
        const int l = cm.xsrc == SIDE_XLO ? -1 - i : i - g.nx;
        if (l < 3) {
            const double* sp = src + src_off(g.nx, g.ny, cm.xsrc) + 3 * ((size_t)(g.ny + 6) * l + r + 3);
            if (sp[0] > 0.0) { c.q1 = sp[0]; c.q2 = sp[1]; c.q3 = sp[2]; return c; }
        }
    }
    if (rm.ysrc >= 0) {
        const int l = rm.ysrc == SIDE_YLO ? -1 - r : r - g.ny;
        if (l < 3) {
            const double* sp = src + src_off(g.nx, g.ny, rm.ysrc) + 3 * ((size_t)g.nx * l + cm.col);
            if (sp[0] > 0.0) { c.q1 = sp[0]; c.q2 = cm.neg2 ? -sp[1] : sp[1]; c.q3 = sp[2]; }
        }
    }
    return c;
}

// End of a step kernel: the running maxima and flags of this block are in the clock; the block that finishes last
// advances the clock (clock_advance) -- no separate clock kernel, no host round trip (PAPER.md:279 lags dt by one step).
// Every thread of the block must call it.
__device__ __forceinline__ bool step_tail(const Grid& g, Clock* clk, double value, int mode, int more) {
    __shared__ int is_last;
    __threadfence();                                                // this thread's atomics before the ticket
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned total = gridDim.x * gridDim.y * gridDim.z;
        is_last = atomicAdd(&clk->ticket, 1u) == total - 1u;
        __threadfence();
    }
    __syncthreads();
    if (is_last && threadIdx.x == 0) clock_advance(g, clk, value, mode, more);
    return is_last;                                                 // block-uniform
}

// Analytic override of a loaded ghost value (same precedence as load_ext: x rule first, then y rule).  Rare path:
// everything by value so that nothing of the caller is forced into local memory.
__device__ __noinline__ double3 apply_sources(Grid g, int xsrc, int ysrc, int col, bool neg2, int i, int r, double t,
                                              double c1, double c2, double c3) {
    Q3 s;
    if (xsrc >= 0 && source_at(g, xsrc, i, r, t, s)) return make_double3(s.q1, s.q2, s.q3);
    if (ysrc >= 0 && source_at(g, ysrc, col, r, t, s))          // col: the (x-mapped) column the y rule is applied on
        return make_double3(s.q1, neg2 ? -s.q2 : s.q2, s.q3);
    return make_double3(c1, c2, c3);
}

// z = (q2/q1, q3/q1) of the one-deep ghost of an intermediate state, from the z of the interior cell next to the
// edge (source step, reading A9): EXTRAP copies, REFLECT negates the normal velocity, SOURCE is analytic inside the
// aperture and EXTRAP outside.  (PERIODIC edges never come here.)
__device__ __noinline__ double2 ghost_z(Grid g, int sd, int i, int r, double t, double z2, double z3) {
    const int kind = g.side[sd].kind;
    if (kind == BC_REFLECT) return sd < 2 ? make_double2(-z2, z3) : make_double2(z2, -z3);
    if (kind == BC_SOURCE) {
        Q3 s;
        if (source_at(g, sd, i, r, t, s)) {
            const double rc = rcp_o1(s.q1);
            return make_double2(s.q2 * rc, s.q3 * rc);
        }
    }
    return make_double2(z2, z3);
}

// Rolling y-state of one interface (the newest one): its cell on the high side, waves, 1/(r.r), and the limiter
// inputs it would take from the interface below it (used if that one is its upwind side).
template <class T> struct YSetT {
    CxT<T> c;
    WvT<T> w;
    T rn1, rn2;
    T pb1, pb2, pb3;
};
using YSet = YSetT<double>;

// Shared-memory layout: ten arrays of double2, one element per column (+ one pad element on each side so that
// tid-1 / tid+1 never clamp).  Every access is [p + constant] from ONE per-thread pointer p = base + 16 (tid+1);
// 128-bit accesses of consecutive columns are bank-conflict free.
//   0 (q1,q2)  1 (q3,hz2)  2 (hz3,-)  3 (al1,s1)  4 (r31,al3)  5 (al2,s2)  6 (r32,-)  7 (m1,m2)  8 (m3,-)  9 (z2,z3)
constexpr int SM_ARRAYS = 10;
template <int BX> __host__ __device__ constexpr int sm_off(int k) { return k * (BX + 2) * 16; }

__device__ __forceinline__ void sts2(char* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }
__device__ __forceinline__ void sts2(char* p, float a, float b) { *reinterpret_cast<float2*>(p) = make_float2(a, b); }
__device__ __forceinline__ double2 lds2(const char* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void sts1(char* p, double a) { *reinterpret_cast<double*>(p) = a; }
__device__ __forceinline__ void sts1(char* p, float a) { *reinterpret_cast<float*>(p) = a; }
__device__ __forceinline__ double lds1(const char* p) { return *reinterpret_cast<const double*>(p); }
template <class T> __device__ __forceinline__ typename Num<T>::T2 ldp(const char* p) { return *reinterpret_cast<const typename Num<T>::T2*>(p); }
template <class T> __device__ __forceinline__ T ld1(const char* p) { return *reinterpret_cast<const T*>(p); }

// Rows of Q^n are prefetched two ticks ahead with cp.async (LDGSTS) into a four-slot ring of shared memory, each
// thread copying and later reading only its own three values -- no barrier needed, no registers held by loads in
// flight, and the compiler cannot sink the loads towards their use.
__device__ __forceinline__ void cp_async8(char* smem_dst, const double* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_elem(char* smem_dst, const double* gsrc) { cp_async8(smem_dst, gsrc); }
__device__ __forceinline__ void cp_async_elem(char* smem_dst, const float* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
template <int BX> __host__ __device__ constexpr int pre_slot_bytes() { return 3 * BX * 8; }

// Block-invariant quantities of a step.
template <class T> struct StepKT {
    double t;
    T lamx, lamy, kapx, kapy, k2;            // k2 = -2 (kapx + kapy)
    T b2, omb2;                              // 2 (beta - 1), 1 - b2
    int j0, j1;                              // rows of output of this chunk: [j0, j1)
    int ylo, ycnt;                           // y-interface ry-1/2 is one the scheme solves iff (unsigned)(ry-ylo) <= ycnt
    bool px, py, any_src, any_refl;
    const double* src;                       // analytic ghost cells of this step (k_step_ws), see src_buffer
};
using StepK = StepKT<double>;

// Per-thread constants and running reductions.
struct ThreadK {
    ColMap cm;
    int i;                                   // column on the ghost-extended mesh
    bool out_col;
    char* p;                                 // this column's element of the shared-memory arrays
    char* pq;                                // this column's element of slot 0 / field 0 of the prefetch ring
    int special;                             // bit 0: fixW, bit 1: fixE (source-step ghosts at the x edges),
                                             // bit 2: ghost column of a REFLECT side, bit 3: of a SOURCE side
    // running reductions (masked by validity at the end)
    double smx, smy;
    int mqx, mdx, mqy, mdy, mxo;             // min high words of q1 / disc in x and y; max |high word| of the output
};

// Carried between ticks besides the two YSets.
struct Carry {
    double s1, s2, s3;                       // Q*(., r-1), left by the previous tick for the y-sweep
    double gp1, gp2, gp3, gf1;               // right-going part (and F~, comp. 1) of the y-interface below the newest one
    double c1, c2, c3, zC2, zC3;             // Q**(r-3) and its z
    double zS2, zS3;                         // z of Q**(r-4)
};

// One tick.  The x-sweep works on row r of Q^n; the y-sweep and the source step run one row behind, on Q*(., ry),
// ry = r-1, which the previous tick left in `cy.s*` -- so each phase between two barriers holds two independent
// instruction streams (x and y) for the scheduler to interleave.
// A: the set of the newest y-interface so far, ry-1/2 - 1 (its cell = Q*(ry-1)); N: on entry its cell still holds
// Q*(ry-2) (from two ticks ago), on exit N is the set of interface ry-1/2 (cell Q*(ry)).
// STEADY: the tick is in the steady part of the march of an interior stretch of rows -- every row it touches is an
// interior row, every pipeline stage holds real data and writes output, no y-edge is near; then all the per-tick
// conditions are known at compile time (the kernel runs the few other ticks of a chunk with STEADY = false).
template <int BX, bool STEADY>
__device__ __forceinline__ void tick(const Grid& g, const StepK& k, ThreadK& th, Carry& cy, const YSet& A, YSet& N, int r,
                                     const double* __restrict__ q1,
                                     const double* __restrict__ q2, const double* __restrict__ q3,
                                     double* __restrict__ o1, double* __restrict__ o2, double* __restrict__ o3) {
    const int ry = r - 1;
    RowMap rm, rm_pre;                                                        // rows r and r+2 (the one to prefetch)
    if (STEADY) {
        rm.row = r; rm.neg3 = false; rm.ysrc = -1;
        rm_pre.row = r + 2;
    } else {
        rm = map_row(g, r);
        rm_pre = map_row(g, r + 2);
    }
    // ---- phase 0: this tick's cell of Q^n (prefetch row r+2); y-cell of Q*(ry) ------------------------------------
    cp_async_wait<1>();                                                       // row r has landed (row r+1 may be in flight)
    double a1, a2, a3;
    {
        const char* ps = th.pq + (r & 3) * pre_slot_bytes<BX>();
        a1 = lds1(ps); a2 = lds1(ps + BX * 8); a3 = lds1(ps + 2 * BX * 8);
        char* pd = th.pq + ((r + 2) & 3) * pre_slot_bytes<BX>();
        const size_t idx = (size_t)rm_pre.row * g.nx + th.cm.col;
        cp_async8(pd, q1 + idx); cp_async8(pd + BX * 8, q2 + idx); cp_async8(pd + 2 * BX * 8, q3 + idx);
        cp_async_commit();
    }
    if (!STEADY && rm.neg3) a3 = -a3;
    if ((th.special & 12) || (!STEADY && rm.ysrc >= 0)) {                     // ghost column of a REFLECT / SOURCE side,
        if (th.special & 4) a2 = -a2;                                         // ghost row of a SOURCE side: rare
        if ((th.special & 8) || rm.ysrc >= 0) {
            const double3 s = apply_sources(g, th.cm.xsrc, rm.ysrc, th.cm.col, th.cm.neg2, th.i, r, k.t, a1, a2, a3);
            a1 = s.x; a2 = s.y; a3 = s.z;
        }
    }
    const bool row_in = STEADY || (unsigned)r < (unsigned)g.ny;
    int tq = 0x7fffffff, td = 0x7fffffff, tqy = 0x7fffffff, tdy = 0x7fffffff;
    const Cx cx = cell_of(a1, a2, a3, tq);
    char* const p = th.p;
    sts2(p + sm_off<BX>(0), cx.q1, cx.q2); sts2(p + sm_off<BX>(1), cx.q3, cx.hz2); sts1(p + sm_off<BX>(2), cx.hz3);
    const double b1o = N.c.q1, b2o = N.c.q2, b3o = N.c.q3;                    // Q*(ry-2), y-form (before N is overwritten)
    N.c = cell_of(cy.s1, cy.s3, cy.s2, tqy);                                  // positions 2,3 switched
    __syncthreads();                                                          // B1: cells (and last tick's z) visible

    // ---- phase 1: x-Riemann at i-1/2 of row r; y-Riemann at ry-1/2 ----------------------------------------------
    Cx L;
    {
        const double2 u0 = lds2(p + sm_off<BX>(0) - 16), u1 = lds2(p + sm_off<BX>(1) - 16);
        L.q1 = u0.x; L.q2 = u0.y; L.q3 = u1.x; L.hz2 = u1.y; L.hz3 = lds1(p + sm_off<BX>(2) - 16);
    }
    double2 zW = lds2(p + sm_off<BX>(9) - 16), zE = lds2(p + sm_off<BX>(9) + 16);   // z of row ry-3, published last tick
    const Wv w = riemann2(L, cx, k.b2, k.omb2, td);
    const double rn1 = rnorm(w.s1, w.r31), rn2 = rnorm(w.s2, w.r32);
    sts2(p + sm_off<BX>(3), w.al1, w.s1); sts2(p + sm_off<BX>(4), w.r31, w.al3); sts2(p + sm_off<BX>(5), w.al2, w.s2);
    sts1(p + sm_off<BX>(6), w.r32);
    N.w = riemann2(A.c, N.c, k.b2, k.omb2, tdy);
    N.rn1 = rnorm(N.w.s1, N.w.r31); N.rn2 = rnorm(N.w.s2, N.w.r32);
    const double d1 = rdot(A.w.s1, A.w.r31, N.w.s1, N.w.r31), d2 = rdot(A.w.s2, A.w.r32, N.w.s2, N.w.r32);
    N.pb1 = A.w.al1 * d1 * N.rn1; N.pb2 = A.w.al2 * d2 * N.rn2; N.pb3 = A.w.al3;      // if A is N's upwind side
    const double hb1 = N.w.al1 * d1 * A.rn1, hb2 = N.w.al2 * d2 * A.rn2;              // if N is A's upwind side
    const Fl G = flux2(A.w, hi_word(A.w.s1) < 0 ? hb1 : A.pb1, hi_word(A.w.s2) < 0 ? hb2 : A.pb2,
                       hi_word(A.w.v) < 0 ? N.w.al3 : A.pb3, k.lamy);
    const double n1 = update_q1(b1o, k.lamy, cy.gp1 + G.m1, cy.gf1, G.ft1);   // Q**(i, ry-2); physical order n1, n2, n3
    const double n3 = fma(-k.lamy, cy.gp2 + G.m2, b2o);
    const double n2 = fma(-k.lamy, cy.gp3 + G.m3, b3o);
    cy.gp1 = G.p1; cy.gp2 = G.p2; cy.gp3 = G.p3; cy.gf1 = G.ft1;
    if (row_in) {
        th.mqx = min(th.mqx, tq); th.mdx = min(th.mdx, td);
        th.smx = dmax(th.smx, fabs(hi_word(w.v) < 0 ? w.s2 : w.s1));          // max(|s1|,|s2|) = |v| + a
    }
    if (STEADY || (unsigned)(ry - k.ylo) <= (unsigned)k.ycnt) {               // y-interface ry-1/2 is one the scheme solves
        th.mqy = min(th.mqy, tqy); th.mdy = min(th.mdy, tdy);
        if (STEADY || (unsigned)ry <= (unsigned)g.ny) th.smy = dmax(th.smy, fabs(hi_word(N.w.v) < 0 ? N.w.s2 : N.w.s1));
    }
    __syncthreads();                                                          // B2: waves visible

    // ---- phase 2: limited fluxes of the x-interface i-1/2 and of the y-interface ry-3/2 (A) ----------------------
    Fl F;
    {
        const char* u1 = p + (hi_word(w.s1) < 0 ? 16 : -16);                  // upwind interface
        const char* u2 = p + (hi_word(w.s2) < 0 ? 16 : -16);
        const char* u3 = p + (hi_word(w.v) < 0 ? 16 : -16);
        const double2 k1 = lds2(u1 + sm_off<BX>(3)), k2 = lds2(u2 + sm_off<BX>(5));
        const double k1r = lds1(u1 + sm_off<BX>(4)), k2r = lds1(u2 + sm_off<BX>(6)), k3 = lds1(u3 + sm_off<BX>(4) + 8);
        const double b1 = k1.x * rdot(k1.y, k1r, w.s1, w.r31) * rn1;
        const double b2 = k2.x * rdot(k2.y, k2r, w.s2, w.r32) * rn2;
        F = flux2(w, b1, b2, k3, k.lamx);
    }
    sts2(p + sm_off<BX>(7), F.m1, F.m2); sts2(p + sm_off<BX>(8), F.m3, F.ft1);
    // source step, x part for row ry-3
    if (th.special & 3) {
        if (th.special & 1) zW = ghost_z(g, SIDE_XLO, -1, ry - 3, k.t, cy.zC2, cy.zC3);
        if (th.special & 2) zE = ghost_z(g, SIDE_XHI, g.nx, ry - 3, k.t, cy.zC2, cy.zC3);
    }
    const double H2 = fma(k.k2, cy.zC2, fma(k.kapx, zE.x + zW.x, cy.c2));
    const double H3 = fma(k.k2, cy.zC3, fma(k.kapx, zE.y + zW.y, cy.c3));
    __syncthreads();                                                          // B3: left-going parts visible

    // ---- phase 3: Q*(i, r) for the next tick; source step (26): publish z of row ry-2, finish row R = ry-3 -------
    {
        const double2 gm = lds2(p + sm_off<BX>(7) + 16);
        const double2 gm3f = lds2(p + sm_off<BX>(8) + 16);
        const double gm3 = gm3f.x;
        cy.s1 = update_q1(a1, k.lamx, F.p1 + gm.x, F.ft1, gm3f.y);
        cy.s2 = fma(-k.lamx, F.p2 + gm.y, a2);
        cy.s3 = fma(-k.lamx, F.p3 + gm3, a3);
    }
    const double rq = rcp_o1(n1);
    const double zN2 = n2 * rq, zN3 = n3 * rq;
    sts2(p + sm_off<BX>(9), zN2, zN3);                                        // read after B1 of the next tick
    const int R = ry - 3;
    if (STEADY || R >= k.j0) {                                                // R < j1 by the loop bound
        double y2 = zN2 + cy.zS2, y3 = zN3 + cy.zS3;
        if (!STEADY && !k.py && (R == 0 || R == g.ny - 1)) {
            double2 lo = make_double2(cy.zS2, cy.zS3), hi = make_double2(zN2, zN3);
            if (R == 0) lo = ghost_z(g, SIDE_YLO, th.i, -1, k.t, cy.zC2, cy.zC3);
            if (R == g.ny - 1) hi = ghost_z(g, SIDE_YHI, th.i, g.ny, k.t, cy.zC2, cy.zC3);
            y2 = hi.x + lo.x; y3 = hi.y + lo.y;
        }
        const double w2 = fma(k.kapy, y2, H2), w3 = fma(k.kapy, y3, H3);
        if (th.out_col) {
            const size_t o = (size_t)R * g.nx + th.i;
            o1[o] = cy.c1; o2[o] = w2; o3[o] = w3;
            th.mxo = max(th.mxo, max(hi_word(cy.c1) & 0x7fffffff, max(hi_word(w2) & 0x7fffffff, hi_word(w3) & 0x7fffffff)));
        }
    }
    cy.zS2 = cy.zC2; cy.zS3 = cy.zC3;
    cy.c1 = n1; cy.c2 = n2; cy.c3 = n3; cy.zC2 = zN2; cy.zC3 = zN3;
}

template <int BX>
__host__ __device__ constexpr int fused_smem_bytes() { return sm_off<BX>(SM_ARRAYS) + 4 * pre_slot_bytes<BX>(); }

// The step kernel.  grid = (strips, chunks); block = BX threads; dynamic shared memory = fused_smem_bytes<BX>().
// rows: rows of output per chunk.
// MINB: blocks per SM the register budget is set for (65536 registers / (BX * MINB) per thread, multiple of 8).
template <int BX, int MINB>
__global__ void __launch_bounds__(BX) __maxnreg__((65536 / (BX * MINB)) / 8 * 8 > 255 ? 255 : (65536 / (BX * MINB)) / 8 * 8)
k_step_fused(Grid g, Clock* clk, const double* __restrict__ q1,
                                                         const double* __restrict__ q2, const double* __restrict__ q3,
                                                         double* __restrict__ o1, double* __restrict__ o2,
                                                         double* __restrict__ o3, int rows, double value, int mode, int more) {
    extern __shared__ __align__(16) char smem[];
    const int tid = threadIdx.x;
    for (int k = tid; k < fused_smem_bytes<BX>() / 8; k += BX) reinterpret_cast<double*>(smem)[k] = 0.0;

    StepK k;
    k.t = clk->t; k.lamx = clk->lamx; k.lamy = clk->lamy; k.kapx = clk->kapx; k.kapy = clk->kapy;
    k.k2 = -2.0 * (k.kapx + k.kapy);
    k.b2 = 2.0 * (g.beta - 1.0); k.omb2 = 1.0 - k.b2;
    k.j0 = (int)blockIdx.y * rows; k.j1 = min(k.j0 + rows, g.ny);
    k.ylo = max(k.j0 - 2, -1); k.ycnt = g.ny + 1 - k.ylo;
    k.px = g.side[SIDE_XLO].kind == BC_PERIODIC; k.py = g.side[SIDE_YLO].kind == BC_PERIODIC;
    k.any_src = g.side[0].kind == BC_SOURCE || g.side[1].kind == BC_SOURCE || g.side[2].kind == BC_SOURCE ||
                g.side[3].kind == BC_SOURCE;
    k.any_refl = g.side[0].kind == BC_REFLECT || g.side[1].kind == BC_REFLECT || g.side[2].kind == BC_REFLECT ||
                 g.side[3].kind == BC_REFLECT;

    ThreadK th;
    th.i = (int)blockIdx.x * (BX - 6) - 3 + tid;
    th.cm = map_column(g, th.i);
    th.special = (!k.px && th.i == 0 ? 1 : 0) | (!k.px && th.i == g.nx - 1 ? 2 : 0) | (th.cm.neg2 ? 4 : 0) |
                 (th.cm.xsrc >= 0 ? 8 : 0);
    th.out_col = tid >= 3 && tid <= BX - 4 && th.i >= 0 && th.i < g.nx;
    th.p = smem + (tid + 1) * 16;
    th.pq = smem + sm_off<BX>(SM_ARRAYS) + tid * 8;
    th.smx = 0.0; th.smy = 0.0;
    th.mqx = th.mdx = th.mqy = th.mdy = 0x7fffffff; th.mxo = 0;

    YSet Y0, Y1;
    Y0.c = {1.0, 0.0, 0.0, 0.0, 0.0};
    Y0.w = {0.0, 1.0, 0.0, 0.0, -1.0, 0.0, 0.0, 0.0};
    Y0.rn1 = Y0.rn2 = 0.5; Y0.pb1 = Y0.pb2 = Y0.pb3 = 0.0;
    Y1 = Y0;
    Carry cy;
    cy.gp1 = cy.gp2 = cy.gp3 = cy.gf1 = 0.0;
    cy.s1 = 1.0; cy.s2 = cy.s3 = 0.0;
    cy.c1 = 1.0; cy.c2 = cy.c3 = cy.zC2 = cy.zC3 = cy.zS2 = cy.zS3 = 0.0;

    int r = k.j0 - 3;
    const int rend = k.j1 + 4;                                     // the y-sweep and the source step run one row behind
    __syncthreads();                                               // (the zero fill above is complete)
    for (int d = 0; d < 2; ++d) {                                  // rows r and r+1 start their way into the ring
        const RowMap rm = map_row(g, r + d);
        const size_t idx = (size_t)rm.row * g.nx + th.cm.col;
        char* pd = th.pq + ((r + d) & 3) * pre_slot_bytes<BX>();
        cp_async8(pd, q1 + idx); cp_async8(pd + BX * 8, q2 + idx); cp_async8(pd + 2 * BX * 8, q3 + idx);
        cp_async_commit();
    }
    // steady ticks: r in [slo, shi] (see tick<>): rows r, r+1 interior; output row r-4 >= j0, away from the y edges
    const int slo = max(k.j0 + 4, k.py ? 0 : 5), shi = min(rend - 1, g.ny - 3);
    while (r < rend && r < slo) {                                  // pipeline fill (and everything, near the y edges)
        tick<BX, false>(g, k, th, cy, Y0, Y1, r, q1, q2, q3, o1, o2, o3);
        const YSet t = Y0; Y0 = Y1; Y1 = t;
        ++r;
    }
    for (; r + 1 <= shi; r += 2) {
        tick<BX, true>(g, k, th, cy, Y0, Y1, r, q1, q2, q3, o1, o2, o3);
        tick<BX, true>(g, k, th, cy, Y1, Y0, r + 1, q1, q2, q3, o1, o2, o3);
    }
    while (r < rend) {
        tick<BX, false>(g, k, th, cy, Y0, Y1, r, q1, q2, q3, o1, o2, o3);
        const YSet t = Y0; Y0 = Y1; Y1 = t;
        ++r;
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
    step_tail(g, clk, value, mode, more);
}

}  // namespace fvnl
