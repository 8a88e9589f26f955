// fvnl_small.cuh -- ALL time steps of a fvnl_step call in ONE launch of ONE thread-block cluster, with the state resident in
// the cluster's DISTRIBUTED SHARED MEMORY, for grids so small that a step is bound by launches and latency, not by
// throughput (BASELINE.json's config C1: 512 x 4 cells x 2000 steps).
//
// Why.  The row-marching step kernel (fvnl_ws.cuh) needs 15 ticks of ~1 us for C1's 4 rows and one launch per step:
// ~20 us per step for 2048 cells.  Here the cells of every sub-step are spread over the threads of up to 16 CTAs on 16
// SMs -- one thread-block cluster, the largest unit of B200 with a hardware barrier (barrier.cluster, ~0.2 us) and with
// load/store access to each other's shared memory -- and the time loop runs INSIDE the kernel:
//     x-sweep (24) on the y-extended mesh   -> cluster barrier
//     y-sweep (25)                          -> cluster barrier
//     source step (26) | a ninth warp combines the partial maxima of all CTAs and advances the CTA's copy of the
//                        clock (the source step does not enter M)                -> cluster barrier
// Q^n, Q* and Q** are three "distributed arrays": the mesh is cut into one TILE per CTA, a CTA computes and stores the cells
// of its tile, and a neighbour's value is a plain load through the cluster's shared-memory window (~200 cycles remote, ~40
// local; ~20 B per cycle and SM), needed for the 2-cell halo of a sweep only.  (History, C1, us per step: state in global
// memory 9.5 -- an L2 round trip is ~700 cycles and a cluster barrier that has to publish global stores ~1.5 us; shared memory
// with blocks of 256 consecutive cells dealt round-robin 7.6 -- every load of the x-sweep remote, half of the CTAs idle in
// the other sub-steps; tiles 5.65.)  HBM is touched twice per CALL: the state is read at the start and written at the end.
// The clock (t, dt, M: PAPER.md:275-279) is kept in every CTA's shared memory -- same inputs, same operations, same values --
// and written back once at the end.
// Arithmetic: the per-cell sub-step functions of the three-pass path (fvnl_unfused.cuh: every thread solves the Riemann
// problems of its own 5-cell stencil; ghost rules and analytic source cells evaluated on load, fvnl_bc.cuh).
#pragma once
#include <cooperative_groups.h>

#include "fvnl_fused.cuh"

namespace fvnl {

constexpr int SMALL_THREADS = 256;
constexpr int SMALL_MAX_CLUSTER = 16;                      // non-portable cluster size (8 is the portable maximum)
constexpr size_t SMALL_MAX_CELLS = 16384;                  // beyond this the row-marching kernel is faster
constexpr int SMALL_MAX_SMEM = 225 * 1024;                 // dynamic shared memory a CTA may ask for (227 KB per SM, some static)

// Cluster barrier between sub-steps.  Everything the sub-steps exchange lives in SHARED memory (the CTA's own or, through the
// cluster window, another CTA's), so what has to be ordered before the arrival are this CTA's shared-memory stores: a CTA-scope
// fence.  cooperative_groups' cluster.sync() releases at cluster scope for ALL memory, which ptxas turns into MEMBAR.ALL.GPU
// (ncu: 8.5 % of the kernel's stall samples).
__device__ __forceinline__ void cluster_sync_shared() {
    __threadfence_block();
    asm volatile("barrier.cluster.arrive.relaxed.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

struct SmallPartial {                                      // what one CTA contributes to the end of a step
    unsigned long long sx, sy;                             // max |s| over its x- / y-interfaces (bit patterns)
    int flags, pad;
};

__device__ __forceinline__ unsigned long long warp_max_bits(double v) {
    unsigned long long b = (unsigned long long)__double_as_longlong(v);
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
        b = other > b ? other : b;
    }
    return b;
}

// How the mesh is spread over the C = Cx x Cy CTAs of the cluster: TILES of W x H cells (Q*, on the y-extended mesh of ny + 4
// rows: W x Hs).  A CTA computes and stores the cells of its own tile, so that a sweep reads the other CTAs' shared memory
// only for its halo (2 cells in the sweep direction), and every CTA has work in every sub-step.  (The first layout dealt
// blocks of 256 consecutive cells round-robin: on C1 every load of the x-sweep was remote -- 30 KB per CTA and step through
// a window that delivers ~20 B per cycle -- and half of the CTAs had no cell in the y-sweep and the source step.)
// Cx starts at C and is halved while tiles would be narrower than 8 cells or more than twice as tall as wide.
struct Tiling {
    int cx_log, cy_log, W, H, Hs;
};
__host__ __device__ inline Tiling small_tiling(int nx, int ny, int C) {
    int cx = C, cy = 1;
    auto cdiv = [](int a, int b) { return (a + b - 1) / b; };
    while (cx > 1 && (cdiv(nx, cx) < 8 || 2 * cdiv(nx, cx) < cdiv(ny, cy))) { cx /= 2; cy *= 2; }
    Tiling t;
    t.cx_log = 0; while ((1 << t.cx_log) < cx) ++t.cx_log;
    t.cy_log = 0; while ((1 << t.cy_log) < cy) ++t.cy_log;
    t.W = cdiv(nx, cx); t.H = cdiv(ny, cy); t.Hs = cdiv(ny + 4, cy);
    return t;
}
// floor(a / b) for 0 <= a < 2^20, 1 <= b: (a + 0.5) / b is never within 0.5 / b of an integer, far more than fp32 rounding.
__device__ __forceinline__ int fdiv(int a, float inv_b) { return __float2int_rd(((float)a + 0.5f) * inv_b); }

// A cell array of `rows` x nx cells in tiles of W x H over the cluster: three planes of `cap` doubles at the same
// shared-memory offset in every CTA; cell (row, col) is element (row % H) W + col % W of CTA (col / W) + Cx (row / H).
struct DistCells {
    double* base;                                          // this CTA's copy (generic address of shared memory)
    int cap, nx, W, H, cx_log;
    float inv_nx, inv_W, inv_H;
    __device__ __forceinline__ const double* at(int row, int col) const {
        const int tx = fdiv(col, inv_W), ty = fdiv(row, inv_H);
        const double* p = base + (row - ty * H) * W + (col - tx * W);
        return cooperative_groups::this_cluster().map_shared_rank(p, (unsigned)(tx + (ty << cx_log)));
    }
    __device__ __forceinline__ const double* where(size_t idx) const {
        const int row = fdiv((int)idx, inv_nx);
        return at(row, (int)idx - row * nx);
    }
    // cell (row, col) as a 32-bit code, owner << 24 | offset in the owner's plane, and the cell behind such a code
    __device__ __forceinline__ unsigned code(int row, int col) const {
        const int tx = fdiv(col, inv_W), ty = fdiv(row, inv_H);
        return (unsigned)((tx + (ty << cx_log)) << 24) | (unsigned)((row - ty * H) * W + (col - tx * W));
    }
    __device__ __forceinline__ Q3 by_code(unsigned code) const {
        const double* p = cooperative_groups::this_cluster().map_shared_rank(base + (code & 0xffffffu), code >> 24);
        Q3 c;
        c.q1 = p[0]; c.q2 = p[cap]; c.q3 = p[2 * cap];
        return c;
    }
    __device__ __forceinline__ Q3 operator()(size_t idx) const {
        const double* p = where(idx);
        Q3 c;
        c.q1 = p[0]; c.q2 = p[cap]; c.q3 = p[2 * cap];
        return c;
    }
    __device__ __forceinline__ void put(size_t idx, const Q3& c) const {        // (idx must be a cell of this CTA's tile)
        const int row = fdiv((int)idx, inv_nx), col = (int)idx - row * nx;
        double* p = base + (row - fdiv(row, inv_H) * H) * W + (col - fdiv(col, inv_W) * W);
        p[0] = c.q1; p[cap] = c.q2; p[2 * cap] = c.q3;
    }
};
__device__ __forceinline__ DistCells make_dist(double* base, int cap, int nx, int W, int H, int cx_log) {
    return DistCells{base, cap, nx, W, H, cx_log, 1.0f / (float)nx, 1.0f / (float)W, 1.0f / (float)H};
}
// Cell number `l` (0 .. W H - 1) of the tile (tx, ty) of such an array with `rows` rows: its index row * nx + col, or -1 when it
// lies outside the mesh (ragged last tiles).
__device__ __forceinline__ int tile_cell(const DistCells& d, int tx, int ty, int rows, int l) {
    const int lr = fdiv(l, d.inv_W), row = ty * d.H + lr, col = tx * d.W + (l - lr * d.W);
    return (lr < d.H && row < rows && col < d.nx) ? row * d.nx + col : -1;
}

// The analytic records of SOURCE sides (1-D), dealt one by one round-robin over the CTAs: record m lives in -- and is
// evaluated by -- CTA m mod C (in blocks of 256 the 30 records of C1's piston were all CTA 0's, whose clock warp then took
// longer over them than the x-sweep it runs beside).
struct DistRecords {
    double* base;
    int cap, logc;
    __device__ __forceinline__ Q3 operator()(size_t idx) const {
        const double* p = cooperative_groups::this_cluster().map_shared_rank(base + (idx >> logc), (unsigned)idx & ((1u << logc) - 1u));
        Q3 c;
        c.q1 = p[0]; c.q2 = p[cap]; c.q3 = p[2 * cap];
        return c;
    }
    __device__ __forceinline__ void put(size_t idx, const Q3& c) const {        // (idx must be one of this CTA's own)
        double* p = base + (idx >> logc);
        p[0] = c.q1; p[cap] = c.q2; p[2 * cap] = c.q3;
    }
};

// One cell of an x-sweep stencil, resolved ONCE before the time loop (a thread computes the same cells in every step): where
// the ghost rules of fvnl_bc.cuh (x rule first, then y rule: load_ext) send the cell -- a pointer into the distributed Q^n,
// the signs a REFLECT edge flips, and whether an analytic SOURCE edge may override it (that depends on t: evaluated per step).
// Resolving it per step cost two thirds of the x-sweep's instructions (ghost-rule branches, integer divisions).
struct StencilCell {
    const double* p;
    int info;                                              // bit 0: neg2, bit 1: neg3, bit 2: an analytic record may override it
    int xrec, yrec;                                        // analytic cell of the x / y SOURCE side: local slot / record (src_record_index), -1: none
};
__device__ __forceinline__ StencilCell resolve_cell(const Grid& g, const DistCells& A, int i, int r) {
    const ColMap cm = map_column(g, i);
    const RowMap rm = map_row(g, r);
    StencilCell e;
    e.p = A.where((size_t)rm.row * g.nx + cm.col);
    e.xrec = e.yrec = -1;                                  // (two ghost layers: l = 0, 1)
    if (cm.xsrc >= 0) e.xrec = (int)src_record_index(g.nx, g.ny, cm.xsrc, cm.xsrc == SIDE_XLO ? -1 - i : i - g.nx, r);
    if (rm.ysrc >= 0) e.yrec = (int)src_record_index(g.nx, g.ny, rm.ysrc, rm.ysrc == SIDE_YLO ? -1 - r : r - g.ny, cm.col);
    e.info = (cm.neg2 ? 1 : 0) | (rm.neg3 ? 2 : 0) | ((e.xrec >= 0 || e.yrec >= 0) ? 4 : 0);
    return e;
}
// The five cells of a stencil: all fifteen loads first (no branch between them, so that they are in flight together: one
// round trip through the cluster's shared-memory window instead of five), then the signs, then -- rare -- the analytic cells.
// `src`: the analytic cells of this step (distributed array of records, q1 <= 0: outside the aperture / not a SOURCE side).
// `src`: the analytic cells of y sides of this step (distributed records); `xs`, `ns`: those of x sides this CTA's threads read,
// in its own shared memory (three planes of ns doubles; StencilCell::xrec is the slot).
__device__ __forceinline__ void load_stencil(const StencilCell* st, int stride, int cap, const DistRecords& src, const double* xs, int ns,
                                             Q3 v[5]) {
    int info[5], any = 0;
#pragma unroll
    for (int e = 0; e < 5; ++e) {
        const StencilCell c = st[e * stride];
        v[e].q1 = c.p[0]; v[e].q2 = c.p[cap]; v[e].q3 = c.p[2 * cap];
        info[e] = c.info;
        any |= c.info;
    }
#pragma unroll
    for (int e = 0; e < 5; ++e) {
        v[e].q2 = (info[e] & 1) ? -v[e].q2 : v[e].q2;
        v[e].q3 = (info[e] & 2) ? -v[e].q3 : v[e].q3;
    }
    if (any & 4) {                                         // a SOURCE edge in reach: same precedence as load_ext
#pragma unroll
        for (int e = 0; e < 5; ++e)
            if (info[e] & 4) {
                const StencilCell c = st[e * stride];
                Q3 a;
                a.q1 = -1.0;
                if (c.xrec >= 0) { a.q1 = xs[c.xrec]; a.q2 = xs[ns + c.xrec]; a.q3 = xs[2 * ns + c.xrec]; }
                if (a.q1 > 0.0) v[e] = a;
                else if (c.yrec >= 0) {
                    a = src((size_t)c.yrec);
                    if (a.q1 > 0.0) {
                        if (c.info & 1) a.q2 = -a.q2;
                        v[e] = a;
                    }
                }
            }
    }
}

// max over the warp of non-negative doubles given as bit patterns: two 32-bit REDUX instead of five shuffle rounds.
__device__ __forceinline__ unsigned long long warp_max_bits_redux(unsigned long long b) {
    const unsigned hi = (unsigned)(b >> 32), lo = (unsigned)b;
    const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
    const unsigned ml = __reduce_max_sync(0xffffffffu, hi == mh ? lo : 0u);
    return ((unsigned long long)mh << 32) | ml;
}

// clock_advance (fvnl_bc.cuh) by a whole warp: the same operations on the same operands -- bitwise the same clock -- but the
// IEEE divisions that do not depend on one another run in different lanes (sx/dx and sy/dy; then lambda_x, lambda_y, kappa_x,
// kappa_y), so that the chain is three divisions long instead of seven.  sx_bits / sy_bits / flags: the step's maxima and
// flag word, the same in every lane.  Lane 0 writes *next.  All 32 lanes must call it.
__device__ __forceinline__ void clock_advance_warp(const Grid& g, const Clock& now, Clock* next, unsigned long long sx_bits,
                                                   unsigned long long sy_bits, int flags, double value, int mode, int more, int lane) {
    const double s = __longlong_as_double((long long)((lane & 1) ? sy_bits : sx_bits));
    const double q = __ddiv_rn(s, (lane & 1) ? g.dy : g.dx);
    const double M = fmax(__shfl_sync(0xffffffffu, q, 0), __shfl_sync(0xffffffffu, q, 1));
    const double dt_old = now.dt;
    const double cfl = __dmul_rn(__dmul_rn(g.c0, dt_old), M);
    int fl = now.flags | flags;
    if (cfl > 1.0) fl |= F_ECFL;
    double dt = dt_old, r = 0.0;
    if (more) {                                            // clock_set_dt
        dt = (mode == 1) ? __ddiv_rn(value, __dmul_rn(g.c0, M)) : value;
        const double num = __dmul_rn(lane < 2 ? g.c0 : g.delta, dt);
        const double den = lane == 0 ? g.dx : lane == 1 ? g.dy : lane == 2 ? __dmul_rn(g.dx, g.dx) : __dmul_rn(g.dy, g.dy);
        r = __ddiv_rn(num, den);
    }
    const double lamx = __shfl_sync(0xffffffffu, r, 0), lamy = __shfl_sync(0xffffffffu, r, 1),
                 kapx = __shfl_sync(0xffffffffu, r, 2), kapy = __shfl_sync(0xffffffffu, r, 3);
    if (lane == 0) {
        *next = now;
        next->last_dt = dt_old;
        next->last_cfl = cfl;
        next->Mprev = M;
        next->t = __dadd_rn(now.t, dt_old);
        next->steps = now.steps + 1;
        next->ticket = 0u;
        next->sx_bits = sx_bits;                           // (as clock_advance leaves them when no step follows)
        next->sy_bits = sy_bits;
        if (more) {
            next->dt = dt; next->lamx = lamx; next->lamy = lamy; next->kapx = kapx; next->kapy = kapy;
            if (__dadd_rn(kapx, kapy) > 0.5) fl |= F_ECFL;
            if (!(dt > 0.0) || not_finite(dt)) fl |= F_ENAN;
            next->sx_bits = 0ull;
            next->sy_bits = 0ull;
        }
        next->flags = fl;
    }
}

// One cell of the source step, resolved once before the time loop (as StencilCell for the x-sweep): where its four neighbours
// live in Q** (for an edge cell: the cell its ghost is made from -- the wrapped one for PERIODIC, itself otherwise), its own
// offset in the CTA's planes of Q** and Q^n, its position and which edges it touches.
struct SrcCell {
    unsigned w, e, s, n;                                   // DistCells::code
    int own;                                               // offset in this CTA's plane; -1: no cell
    short i, j;
    int edge;                                              // bit 0: x-lo, 1: x-hi, 2: y-lo, 3: y-hi
    int xslot;                                             // local slot of the x side's analytic ghost cell, -1: none
};

// Local slots for the analytic cells of x sides a CTA's threads read: per row of its Q* tile at most three ghost cells on each
// side (columns -2, -1 from column 0's stencil, -1 from column 1's; duplicates get slots of their own), plus the source step's.
__host__ __device__ inline int small_xslots(const Tiling& tl) { return (6 * tl.Hs + 2 * tl.H + 3) & ~3; }
// Doubles per plane and CTA; dynamic shared memory of the kernel.
__host__ __device__ inline int small_round(int n) { return (n + SMALL_THREADS - 1) / SMALL_THREADS * SMALL_THREADS; }
__host__ __device__ inline int small_cap_records(size_t n, int C) { return (int)((n + C - 1) / C + 1) & ~1; }
__host__ __device__ inline size_t small_smem_bytes(int nx, int ny, int C, bool has_src) {
    const Tiling tl = small_tiling(nx, ny, C);
    const size_t cap = small_round(tl.W * tl.H), cap_star = small_round(tl.W * tl.Hs);
    const size_t cap_src = has_src ? small_cap_records(src_off(nx, ny, 4) / 3, C) : 0;   // two buffers (this / the next step)
    const size_t ns = has_src ? small_xslots(tl) : 0;
    return 8 * 3 * (2 * cap + cap_star + 2 * cap_src + 2 * ns) + 5 * cap_star * sizeof(StencilCell) + cap * sizeof(SrcCell) + 4 * ns;
}

// grid = cluster = C = 2^logc CTAs of SMALL_THREADS + 32 threads: SMALL_THREADS compute threads and one warp that ends the
// step (clock) while the compute warps run the source step, which does not enter M.  Dynamic shared memory =
// small_smem_bytes(nx, ny, C, has_src).  q1..q3: the state in global memory (in and out).  The clock must hold dt of the first
// step (k_clock_begin) on entry.
__global__ void __launch_bounds__(SMALL_THREADS + 32) k_steps_cluster(Grid g, Clock* clk, double* q1, double* q2, double* q3,
                                                                     int logc, long long nsteps, double value, int mode) {
    namespace cg = cooperative_groups;
    cg::cluster_group cl = cg::this_cluster();
    extern __shared__ __align__(16) double small_mem[];
    const unsigned rank = cl.block_rank(), C = cl.num_blocks();
    __shared__ SmallPartial part[2];                       // by step parity: read by the other CTAs while the next step runs
    __shared__ Clock ck[2];                                // by step parity: the clock warp writes the next step's
    const int tid = threadIdx.x, lane = tid & 31;
    const bool clock_warp = tid >= SMALL_THREADS;
    const int nx = g.nx, ny = g.ny;
    const Tiling tl = small_tiling(nx, ny, (int)C);
    const int tx = (int)rank & ((1 << tl.cx_log) - 1), ty = (int)rank >> tl.cx_log;      // this CTA's tile
    const int cap = small_round(tl.W * tl.H), cap_star = small_round(tl.W * tl.Hs);
    const int rounds = cap / SMALL_THREADS, rounds_star = cap_star / SMALL_THREADS;
    const DistCells A = make_dist(small_mem, cap, nx, tl.W, tl.H, tl.cx_log);                              // Q^n (and Q^{n+1})
    const DistCells S = make_dist(small_mem + 3 * cap, cap_star, nx, tl.W, tl.Hs, tl.cx_log);              // Q*, y-extended
    const DistCells B = make_dist(small_mem + 3 * cap + 3 * cap_star, cap, nx, tl.W, tl.H, tl.cx_log);     // Q**
    const bool has_src = g.src != nullptr;                                     // (fvnl_step sets it when a side is a SOURCE)
    const int nrec = (int)(src_off(nx, ny, 4) / 3), cap_src = has_src ? small_cap_records(nrec, C) : 0;
    double* const src_mem = small_mem + 6 * cap + 3 * cap_star;                // analytic cells of step n: buffer n & 1
    StencilCell* const stencil = reinterpret_cast<StencilCell*>(src_mem + 6 * cap_src);                // [round k][cell e][thread]
    SrcCell* const stab = reinterpret_cast<SrcCell*>(stencil + 5 * cap_star);                          // [round k][thread]
    const int ns = has_src ? small_xslots(tl) : 0;         // local slots: the analytic cells of x sides this CTA's threads read
    double* const xs_mem = reinterpret_cast<double*>(stab + cap);                                      // [buffer][3][ns]
    int* const slot_rec = reinterpret_cast<int*>(xs_mem + 6 * ns);                                     // record of a slot
    __shared__ int nslots;
    auto new_slot = [&](int rec) {                         // (set-up only)
        const int sl = atomicAdd(&nslots, 1);
        if (sl >= ns) return -1;                           // cannot happen (small_xslots bounds the count)
        slot_rec[sl] = rec;
        return sl;
    };
    // The analytic cells of a step (two ghost layers of every SOURCE side, (41) / (43) / piston at t_n) are evaluated ONE STEP
    // AHEAD -- t_{n+1} = t_n + dt_n is known when step n starts, PAPER.md:279 -- by the clock warp, which idles during the
    // sweeps, each CTA the records it stores; the sweeps and the source step only load them.
    auto make_records = [&](int buf, double t, int who, int nthreads) {
        const DistRecords R{src_mem + 3 * cap_src * buf, cap_src, logc};
        for (int sd = 2; sd < 4; ++sd) {                   // y sides; only the records of SOURCE sides exist for the readers
            if (g.side[sd].kind != BC_SOURCE) continue;
            const int first = (int)(src_off(nx, ny, sd) / 3), cnt = (int)(src_side_doubles(nx, ny, sd) / 3);
            const int per = sd < 2 ? ny + 6 : nx;          // records per ghost layer (layout of Grid::src, fvnl_bc.cuh)
            for (int m = first + (((int)rank - first) & ((int)C - 1)) + (int)C * who; m < first + cnt; m += (int)C * nthreads) {
                const int layer = (m - first) / per, pos = (m - first) - layer * per;
                Q3 c;
                bool in;
                if (sd < 2) in = source_at(g, sd, sd == SIDE_XLO ? -1 - layer : nx + layer, pos - 3, t, c);
                else in = source_at(g, sd, pos, sd == SIDE_YLO ? -1 - layer : ny + layer, t, c);
                if (!in) { c.q1 = -1.0; c.q2 = c.q3 = 0.0; }
                R.put(m, c);
            }
        }
    };
    // ... and the x sides' in the CTA that reads them (its slots), so that the edge tile's loads stay in its own shared memory
    auto make_xslots = [&](int buf, double t, int who, int nthreads) {
        double* xs = xs_mem + 3 * ns * buf;
        const int first1 = (int)(src_off(nx, ny, 1) / 3);
        for (int sl = who; sl < nslots; sl += nthreads) {
            const int m = slot_rec[sl], sd = m >= first1 ? 1 : 0, r = m - (sd ? first1 : 0);
            const int layer = r / (ny + 6), pos = r - layer * (ny + 6);
            Q3 c;
            if (!source_at(g, sd, sd == SIDE_XLO ? -1 - layer : nx + layer, pos - 3, t, c)) { c.q1 = -1.0; c.q2 = c.q3 = 0.0; }
            xs[sl] = c.q1; xs[ns + sl] = c.q2; xs[2 * ns + sl] = c.q3;
        }
    };
    if (tid == 0) { nslots = 0; ck[0] = *clk; part[0].sx = part[0].sy = part[1].sx = part[1].sy = 0ull; part[0].flags = part[1].flags = 0; }
    __syncthreads();                                       // (ck[0])
    if (!clock_warp) {
        for (int k = 0; k < rounds; ++k) {
            const int m = tile_cell(A, tx, ty, ny, k * SMALL_THREADS + tid);
            if (m >= 0) {
                Q3 c;
                c.q1 = q1[m]; c.q2 = q2[m]; c.q3 = q3[m];
                A.put(m, c);
            }
        }
        const bool px = g.side[SIDE_XLO].kind == BC_PERIODIC, py = g.side[SIDE_YLO].kind == BC_PERIODIC;
        for (int k = 0; k < rounds; ++k) {                 // the source step's cells (same choices as source_step_cell)
            const int m = tile_cell(A, tx, ty, ny, k * SMALL_THREADS + tid);
            SrcCell c;
            c.own = -1; c.w = c.e = c.s = c.n = 0u; c.i = c.j = 0; c.edge = 0; c.xslot = -1;
            if (m >= 0) {
                const int j = m / nx, i = m - j * nx;
                const bool xlo = i == 0, xhi = i == nx - 1, ylo = j == 0, yhi = j == ny - 1;
                c.own = (int)(B.code(j, i) & 0xffffffu);
                c.w = B.code(j, xlo ? (px ? nx - 1 : i) : i - 1);
                c.e = B.code(j, xhi ? (px ? 0 : i) : i + 1);
                c.s = B.code(ylo ? (py ? ny - 1 : j) : j - 1, i);
                c.n = B.code(yhi ? (py ? 0 : j) : j + 1, i);
                c.i = (short)i; c.j = (short)j;
                c.edge = (xlo ? 1 : 0) | (xhi ? 2 : 0) | (ylo ? 4 : 0) | (yhi ? 8 : 0);
                const int sd = xlo ? SIDE_XLO : SIDE_XHI;
                if ((xlo || xhi) && g.side[sd].kind == BC_SOURCE) c.xslot = new_slot((int)src_record_index(nx, ny, sd, 0, j));
            }
            stab[k * SMALL_THREADS + tid] = c;
        }
        for (int k = 0; k < rounds_star; ++k) {
            const int m = tile_cell(S, tx, ty, ny + 4, k * SMALL_THREADS + tid);
            if (m >= 0) {
                const int row = m / nx, i = m - row * nx;
#pragma unroll
                for (int e = 0; e < 5; ++e) {
                    StencilCell c = resolve_cell(g, A, i - 2 + e, row - 2);
                    if (c.xrec >= 0) c.xrec = new_slot(c.xrec);
                    stencil[(k * 5 + e) * SMALL_THREADS + tid] = c;
                }
            }
        }
    }
    __syncthreads();                                       // (the slots are allocated)
    if (has_src && !clock_warp) {                          // the analytic cells of the first step
        make_records(0, ck[0].t, tid, SMALL_THREADS);
        make_xslots(0, ck[0].t, tid, SMALL_THREADS);
    }
    cl.sync();
    for (long long step = 0; step < nsteps; ++step) {
        SmallPartial* mine = &part[step & 1];
        const Clock& now = ck[step & 1];
        const DistRecords SRC{src_mem + 3 * cap_src * (int)(step & 1), cap_src, logc};
        const double* xs = xs_mem + 3 * ns * (int)(step & 1);
        if (clock_warp && has_src && step + 1 < nsteps) {
            make_xslots((int)((step + 1) & 1), __dadd_rn(now.t, now.dt), lane, 32);
            make_records((int)((step + 1) & 1), __dadd_rn(now.t, now.dt), lane, 32);
        }
        if (!clock_warp) {                                 // ---- x-sweep (24) on the y-extended mesh
            const double lamx = now.lamx;
            int flags = 0;
            double sx = 0.0;
            for (int k = 0; k < rounds_star; ++k) {
                const int m = tile_cell(S, tx, ty, ny + 4, k * SMALL_THREADS + tid);
                if (m < 0) continue;
                Q3 v[5];
                load_stencil(stencil + (size_t)k * 5 * SMALL_THREADS + tid, SMALL_THREADS, cap, SRC, xs, ns, v);
                const int row = fdiv(m, S.inv_nx);
                xsweep_stencil(g, lamx, v, S, m - row * nx, row - 2, sx, flags);
            }
            const unsigned long long bx = warp_max_bits(sx);
            const int f = __reduce_or_sync(0xffffffffu, flags);
            if (lane == 0) {
                if (bx) atomicMax(&mine->sx, bx);
                if (f) atomicOr(&mine->flags, f);
            }
        }
        cluster_sync_shared();
        if (!clock_warp) {                                 // ---- y-sweep (25)
            const double lamy = now.lamy;
            int flags = 0;
            double sy = 0.0;
            for (int k = 0; k < rounds; ++k) {
                const int m = tile_cell(B, tx, ty, ny, k * SMALL_THREADS + tid);
                if (m < 0) continue;
                const int row = fdiv(m, B.inv_nx);
                ysweep_cell(g, lamy, S, B, m - row * nx, row, sy, flags);
            }
            const unsigned long long by = warp_max_bits(sy);
            const int f = __reduce_or_sync(0xffffffffu, flags);
            if (lane == 0) {
                if (by) atomicMax(&mine->sy, by);
                if (f) atomicOr(&mine->flags, f);
            }
        }
        cluster_sync_shared();
        if (!clock_warp) {                                 // ---- source step (26)
            const double kapx = now.kapx, kapy = now.kapy;
            auto ghost = [&](int sd, const Q3& inner, int pos, int xslot) {     // ghost_of, analytic cells from the records
                const int kind = g.side[sd].kind;
                Q3 c = inner;
                if (kind == BC_REFLECT) {
                    if (sd < 2) c.q2 = -c.q2; else c.q3 = -c.q3;
                } else if (kind == BC_SOURCE) {
                    Q3 a;
                    if (sd < 2) { a.q1 = xs[xslot]; a.q2 = xs[ns + xslot]; a.q3 = xs[2 * ns + xslot]; }
                    else a = SRC(src_record_index(nx, ny, sd, 0, pos));
                    if (a.q1 > 0.0) c = a;
                }
                return c;
            };
            for (int k = 0; k < rounds; ++k) {
                const SrcCell sc = stab[k * SMALL_THREADS + tid];
                if (sc.own < 0) continue;
                const double* pc = B.base + sc.own;        // five independent loads, then -- rare -- the ghost rules
                Q3 c;
                c.q1 = pc[0]; c.q2 = pc[cap]; c.q3 = pc[2 * cap];
                Q3 w = B.by_code(sc.w), e = B.by_code(sc.e), s = B.by_code(sc.s), n = B.by_code(sc.n);
                if (sc.edge) {
                    if (sc.edge & 1) w = ghost(SIDE_XLO, w, sc.j, sc.xslot);
                    if (sc.edge & 2) e = ghost(SIDE_XHI, e, sc.j, sc.xslot);
                    if (sc.edge & 4) s = ghost(SIDE_YLO, s, sc.i, -1);
                    if (sc.edge & 8) n = ghost(SIDE_YHI, n, sc.i, -1);
                }
                const Q3 o = source_step_values(c, w, e, s, n, kapx, kapy);
                double* pa = A.base + sc.own;
                pa[0] = o.q1; pa[cap] = o.q2; pa[2 * cap] = o.q3;
            }
        } else {                                           // ---- end of the step: M_n, nu_n, t_{n+1}, dt_{n+1} (clock_advance)
            unsigned long long bx = 0ull, by = 0ull;       // lane r fetches the partial result of CTA r
            int f = 0;
            if (lane < (int)C) {
                const SmallPartial* p = cl.map_shared_rank(mine, lane);
                bx = p->sx; by = p->sy; f = p->flags;
            }
            bx = warp_max_bits_redux(bx);
            by = warp_max_bits_redux(by);
            f = __reduce_or_sync(0xffffffffu, f);
            clock_advance_warp(g, now, &ck[(step + 1) & 1], bx, by, f, value, mode, step + 1 < nsteps ? 1 : 0, lane);
            if (lane == 0) {
                SmallPartial* other = &part[(step + 1) & 1];               // (last read before the previous cluster barrier)
                other->sx = other->sy = 0ull; other->flags = 0;
            }
        }
        cluster_sync_shared();
    }
    if (!clock_warp)
        for (int k = 0; k < rounds; ++k) {
            const int m = tile_cell(A, tx, ty, ny, k * SMALL_THREADS + tid);
            if (m >= 0) {
                const Q3 c = A(m);
                q1[m] = c.q1; q2[m] = c.q2; q3[m] = c.q3;
            }
        }
    if (rank == 0 && tid == 0) *clk = ck[nsteps & 1];
    cl.sync();                                             // no CTA leaves while another may still read its shared memory
}

}  // namespace fvnl
