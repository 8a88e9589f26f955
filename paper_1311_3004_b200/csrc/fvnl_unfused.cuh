// fvnl_unfused.cuh -- three-pass form of the step: x-sweep, y-sweep and source step as separate kernels, one thread
// per cell, every thread solving the Riemann problems of its own 5-cell stencil (4x redundant).  It exists as the
// measured "what fusion buys" comparison point (144 B/cell-update of HBM traffic) and as the
// second, independently structured GPU implementation the fused kernel is cross-checked against bit by bit in
// tests/.  The product default is the fused kernel (fvnl_fused.cuh); this path is opt-in (FVNL_KERNEL_UNFUSED).
#pragma once
#include "fvnl_bc.cuh"

namespace fvnl {

// Block-wide max of non-negative doubles -> atomicMax on the bit pattern (order preserving for x >= 0).
__device__ __forceinline__ void block_max_to(unsigned long long* slot, double v) {
    unsigned long long b = (unsigned long long)__double_as_longlong(v);
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
        b = other > b ? other : b;
    }
    __shared__ unsigned long long red[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) red[wid] = b;
    __syncthreads();
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        b = lane < nw ? red[lane] : 0ull;
        for (int o = 16; o > 0; o >>= 1) {
            const unsigned long long other = __shfl_xor_sync(0xffffffffu, b, o);
            b = other > b ? other : b;
        }
        if (lane == 0 && b != 0ull) atomicMax(slot, b);
    }
}

__device__ __forceinline__ void block_flags_to(int* slot, int f) {
    f = __reduce_or_sync(0xffffffffu, f);
    if ((threadIdx.x & 31) == 0 && f) atomicOr(slot, f);
}

// (27) for the middle cell of a 5-cell stencil c[0..4] in x-form.  Returns Q* of c[2]; `sl` / `sr`: the speeds of
// its left / right interface for M.
__device__ __forceinline__ Q3 sweep_cell(const CellX c[5], double lam, double beta2m2, double& sl, double& sr, int& flags) {
    Waves w[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) w[k] = riemann_x(c[k], c[k + 1], beta2m2, flags);
    Flux3 F[2];
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const Waves& k = w[1 + e];
        const Waves& lo = w[e];
        const Waves& hi = w[2 + e];
        const bool u1 = k.s1 > 0.0, u2 = k.s2 > 0.0, u3 = k.s3 > 0.0;      // upwind interface is k-1
        F[e] = interface_flux(k, u1 ? lo.al1 : hi.al1, u1 ? lo.s1 : hi.s1, u1 ? lo.r31 : hi.r31,
                              u2 ? lo.al2 : hi.al2, u2 ? lo.s2 : hi.s2, u2 ? lo.r32 : hi.r32,
                              u3 ? lo.al3 : hi.al3, lam);
    }
    sl = max_speed(w[1]);
    sr = max_speed(w[2]);
    Q3 o;
    {   // density: rounded where (27) rounds, PAPER.md:161 (see update_q1 in fvnl_pair.cuh)
        const double s2 = __dsub_rn(F[1].ft1, F[0].ft1), s1 = __dsub_rn(F[0].p1 + F[1].m1, s2);
        o.q1 = __dsub_rn(__dsub_rn(c[2].q1, __dmul_rn(lam, s1)), __dmul_rn(lam, s2));
    }
    o.q2 = fma(-lam, F[0].p2 + F[1].m2, c[2].q2);
    o.q3 = fma(-lam, F[0].p3 + F[1].m3, c[2].q3);
    if (not_finite(o.q1) || not_finite(o.q2) || not_finite(o.q3)) flags |= F_ENAN;
    return o;
}

// ---- one cell of each sub-step ---------------------------------------------------------------------------------------
// Written against "cells" (a callable idx -> Q3) and "out" (put(idx, Q3)) so that the same arithmetic serves the three-pass
// kernels below (planes in global memory) and the small-grid cluster kernel (fvnl_small.cuh: distributed shared memory).
// O2: Q*(i, r) of the x-sweep (24) on the y-extended mesh (row r in -2 .. ny+1 is stored at r + 2 of star).
// v[0..4]: the cells i-2 .. i+2 of row r of the ghost-extended mesh.
template <class Out>
__device__ __forceinline__ void xsweep_stencil(const Grid& g, double lam, const Q3 v[5], const Out& star, int i, int r, double& smax,
                                               int& flags) {
    CellX c[5];
    int f = 0;
#pragma unroll
    for (int k = 0; k < 5; ++k) c[k] = make_cell(v[k].q1, v[k].q2, v[k].q3, f);
    double sl, sr;
    const Q3 o = sweep_cell(c, lam, 2.0 * (g.beta - 1.0), sl, sr, f);
    star.put((size_t)(r + 2) * g.nx + i, o);
    if (r >= 0 && r < g.ny) { smax = fmax(smax, fmax(sl, sr)); flags |= f; }      // ghost rows do not enter M (O5)
}
template <class Cells, class Out>
__device__ __forceinline__ void xsweep_cell(const Grid& g, double t, double lam, const Cells& q, const Out& star, int i, int r,
                                            double& smax, int& flags) {
    Q3 v[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) v[k] = load_ext(g, q, i - 2 + k, r, t);
    xsweep_stencil(g, lam, v, star, i, r, smax, flags);
}

// O3: Q**(i, j) of the y-sweep (25) of star with positions 2 and 3 switched.
template <class Cells, class Out>
__device__ __forceinline__ void ysweep_cell(const Grid& g, double lam, const Cells& star, const Out& out, int i, int j,
                                            double& smax, int& flags) {
    CellX c[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const Q3 v = star((size_t)(j + k) * g.nx + i);               // star row (j-2+k) is stored at j+k
        c[k] = make_cell(v.q1, v.q3, v.q2, flags);
    }
    double sl, sr;
    const Q3 o = sweep_cell(c, lam, 2.0 * (g.beta - 1.0), sl, sr, flags);
    Q3 w;
    w.q1 = o.q1; w.q2 = o.q3; w.q3 = o.q2;
    out.put((size_t)j * g.nx + i, w);
    smax = fmax(smax, fmax(sl, sr));
}

// O4: source step (26): q^m += kap_x d2x(q^m/q^1) + kap_y d2y(q^m/q^1), m = 2, 3 (readings A1, A2), from
// the cell and its four neighbours (ghost rule already applied).
__device__ __forceinline__ Q3 source_step_values(const Q3& c, const Q3& w, const Q3& e, const Q3& s, const Q3& n, double kx, double ky) {
    const double rc = 1.0 / c.q1, rw = 1.0 / w.q1, re = 1.0 / e.q1, rs = 1.0 / s.q1, rn = 1.0 / n.q1;
    const double z2 = c.q2 * rc, z3 = c.q3 * rc;
    const double lx2 = (e.q2 * re + w.q2 * rw) - 2.0 * z2, ly2 = (n.q2 * rn + s.q2 * rs) - 2.0 * z2;
    const double lx3 = (e.q3 * re + w.q3 * rw) - 2.0 * z3, ly3 = (n.q3 * rn + s.q3 * rs) - 2.0 * z3;
    Q3 o;
    o.q1 = c.q1;
    o.q2 = fma(ky, ly2, fma(kx, lx2, c.q2));
    o.q3 = fma(ky, ly3, fma(kx, lx3, c.q3));
    return o;
}
// `ghost(sd, inner, i, r)`: the one-deep ghost cell of side sd at (i, r) made from the loaded cell `inner` (ghost_of).
template <class Cells, class Out, class Ghost>
__device__ __forceinline__ void source_step_cell(const Grid& g, double kx, double ky, const Cells& at_idx, const Out& out,
                                                 const Ghost& ghost, int i, int j) {
    auto at = [&](int ii, int jj) { return at_idx((size_t)jj * g.nx + ii); };
    const bool px = g.side[SIDE_XLO].kind == BC_PERIODIC, py = g.side[SIDE_YLO].kind == BC_PERIODIC;
    // the five loads first, independent of one another (an edge cell loads the cell its ghost is made from: the wrapped one
    // for PERIODIC, itself otherwise), then the ghost rule on the loaded value -- rare, and the loads are all in flight by then
    const bool xlo = i == 0, xhi = i == g.nx - 1, ylo = j == 0, yhi = j == g.ny - 1;
    const Q3 c = at(i, j);
    Q3 w = at(xlo ? (px ? g.nx - 1 : i) : i - 1, j);
    Q3 e = at(xhi ? (px ? 0 : i) : i + 1, j);
    Q3 s = at(i, ylo ? (py ? g.ny - 1 : j) : j - 1);
    Q3 n = at(i, yhi ? (py ? 0 : j) : j + 1);
    if (xlo) w = ghost(SIDE_XLO, w, -1, j);
    if (xhi) e = ghost(SIDE_XHI, e, g.nx, j);
    if (ylo) s = ghost(SIDE_YLO, s, i, -1);
    if (yhi) n = ghost(SIDE_YHI, n, i, g.ny);
    out.put((size_t)j * g.nx + i, source_step_values(c, w, e, s, n, kx, ky));
}

// O2 as a kernel.  grid.y = ny+4.
__global__ void __launch_bounds__(256) k_xsweep_unfused(Grid g, Clock* clk, const double* __restrict__ q1,
                                                        const double* __restrict__ q2, const double* __restrict__ q3,
                                                        double* __restrict__ s1, double* __restrict__ s2,
                                                        double* __restrict__ s3) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int r = (int)blockIdx.y - 2;
    int flags = 0;
    double smax = 0.0;
    if (i < g.nx) xsweep_cell(g, clk->t, clk->lamx, PlaneCells{q1, q2, q3}, PlaneOut{s1, s2, s3}, i, r, smax, flags);
    block_max_to(&clk->sx_bits, smax);
    block_flags_to(&clk->flags, flags);
}

__global__ void __launch_bounds__(256) k_ysweep_unfused(Grid g, Clock* clk, const double* __restrict__ s1,
                                                        const double* __restrict__ s2, const double* __restrict__ s3,
                                                        double* __restrict__ o1, double* __restrict__ o2,
                                                        double* __restrict__ o3) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    int flags = 0;
    double smax = 0.0;
    if (i < g.nx) ysweep_cell(g, clk->lamy, PlaneCells{s1, s2, s3}, PlaneOut{o1, o2, o3}, i, blockIdx.y, smax, flags);
    block_max_to(&clk->sy_bits, smax);
    block_flags_to(&clk->flags, flags);
}

__global__ void __launch_bounds__(256) k_source_unfused(Grid g, const Clock* clk, const double* __restrict__ a1,
                                                        const double* __restrict__ a2, const double* __restrict__ a3,
                                                        double* __restrict__ o1, double* __restrict__ o2,
                                                        double* __restrict__ o3) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const double t = clk->t;
    auto ghost = [&](int sd, const Q3& inner, int gi, int gr) { return ghost_of(g, sd, inner, gi, gr, t); };
    if (i < g.nx) source_step_cell(g, clk->kapx, clk->kapy, PlaneCells{a1, a2, a3}, PlaneOut{o1, o2, o3}, ghost, i, blockIdx.y);
}

}  // namespace fvnl
