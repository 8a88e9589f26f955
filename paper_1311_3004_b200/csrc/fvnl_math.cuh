// fvnl_math.cuh -- per-interface arithmetic of the arXiv 1311.3004 finite-volume step, fp64, sm_100a.
//
// Everything here is register arithmetic shared by the sweep kernels.  "PAPER.md:<line>" cites the paper text.
// The formulation is algebraically the paper's (Roe matrix of the arithmetic-mean primitive state, PAPER.md:218-245;
// waves/fluctuations (28),(29); MC-limited correction (30)) but arranged for
// the FP64 pipe of B200, which is the binding unit of this path:
//   * one reciprocal per cell (1/q1) and per interface (1/Zbar1), one rsqrt per interface (a and 1/a),
//     all as MUFU seed + one third-order Newton step (3 / 5 DFMA), no slow paths: arguments are O(1);
//   * limiter without the division theta = (W_K.W_k)/(W_k.W_k): phi(theta) alpha_k is the homogeneous
//     function mc(alpha_k, alpha_K C/R) with C = r_K.r_k, R = r_k.r_k; the third wave has r = (0,0,1), C = R = 1;
//   * sign handling (max(s,0), |s|, copysign) with integer operations on the high word, which run on the
//     ALU pipe instead of the FP64 pipe.
#pragma once
#include <cuda_runtime.h>

namespace fvnl {

// ---- flag bits (include/fvnl.h) --------------------------------------------------------------------------------
enum { F_ECFL = 16, F_ENONREAL = 32, F_ENONPOS = 64, F_ENAN = 128 };

__device__ __forceinline__ int hi_word(double x) { return __double2hiint(x); }

// 1/x for x of order one: MUFU.RCP64H seed (relative error e ~ 2^-20) and y (1 + e + e^2): error e^3.
__device__ __forceinline__ double rcp_o1(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

// 1/sqrt(x) for x of order one: MUFU.RSQ64H seed and y (1 + e/2 + 3 e^2/8), e = 1 - x y^2.
__device__ __forceinline__ double rsqrt_o1(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    const double q = e * p;
    return fma(y, q, y);
}

// max(s,0) and min(s,0) through the sign bit (ALU pipe).
__device__ __forceinline__ double pos_part(double s) { return hi_word(s) < 0 ? 0.0 : s; }
__device__ __forceinline__ double neg_part(double s) { return hi_word(s) < 0 ? s : 0.0; }

// x with its sign flipped when `sgn` is negative (sign-bit xor, ALU pipe).
__device__ __forceinline__ double xor_sign(double x, double sgn) {
    return __hiloint2double(__double2hiint(x) ^ (__double2hiint(sgn) & 0x80000000), __double2loint(x));
}

// Half of phi(b/a) a for the MC limiter phi(theta) = max(0, min((1+theta)/2, 2, 2 theta)):
//   phi(b/a) a = 2 sgn(a) max(0, min((|a| + B)/4, |a|, B)),  B = sgn(a) b.      a = 0 gives 0 (reading A5).
__device__ __forceinline__ double mc_half(double a, double b) {
    const double A = fabs(a);
    const double B = xor_sign(b, a);
    const double m = fmin(A, B);
    const double q = 0.25 * (A + B);
    const double r = fmax(fmin(m, q), 0.0);
    return xor_sign(r, a);
}

// Per-cell quantities a sweep needs from a cell in x-form (q2 = normal momentum, q3 = transverse momentum):
// the conserved values and half of the primitive velocities z2 = q2/q1, z3 = q3/q1.
struct CellX {
    double q1, q2, q3, hz2, hz3;
};

__device__ __forceinline__ CellX make_cell(double q1, double q2, double q3, int& flags) {
    CellX c;
    c.q1 = q1; c.q2 = q2; c.q3 = q3;
    if (hi_word(q1) <= 0 && !(q1 > 0.0)) flags |= F_ENONPOS;       // q1 <= 0 (or NaN with sign): rare path
    const double hr = 0.5 * rcp_o1(q1);
    c.hz2 = q2 * hr;
    c.hz3 = q3 * hr;
    return c;
}

// Riemann solution at one interface in x-form.  Waves W1 = al1 (1, s1, r31), W2 = al2 (1, s2, r32),
// W3 = (0, 0, al3) with speed s3 = v  (eigenvectors derived in DESIGN.md).
struct Waves {
    double al1, s1, r31, al2, s2, r32, al3, s3;
};

__device__ __forceinline__ Waves riemann_x(const CellX& L, const CellX& R, double beta2m2, int& flags) {
    Waves w;
    const double D1 = R.q1 - L.q1, D2 = R.q2 - L.q2, D3 = R.q3 - L.q3;
    const double Zb1 = fma(0.5, D1, L.q1);                       // (q1L + q1R)/2
    const double Zb2 = L.hz2 + R.hz2;
    const double Zb3 = L.hz3 + R.hz3;
    const double Phi = fma(beta2m2, Zb1, 1.0 - beta2m2);         // 1 + 2(beta-1)(Zb1-1)
    const double u = rcp_o1(Zb1);
    const double v = Zb2 * u;                                    // (34)
    const double wv = Zb3 * u;
    const double tt = fma(-2.0, Zb2, v);                         // v - 2 Zb2
    const double disc = fma(v, tt, Phi);                         // v^2 - 2 Zb2^2/Zb1 + Phi   (32),(33)
    if (hi_word(disc) < 0) flags |= F_ENONREAL;
    const double ra = rsqrt_o1(disc);
    const double a = disc * ra;
    w.s1 = v + a;
    w.s2 = v - a;
    w.s3 = v;
    const double hra = 0.5 * ra;
    w.al1 = fma(-w.s2, D1, D2) * hra;                            // (D2 - s2 D1)/(2a)
    w.al2 = D1 - w.al1;                                          // (s1 D1 - D2)/(2a)
    const double wra = wv * ra;
    w.r31 = wra * (tt + a);                                      //  w (s1 - 2 Zb2)/a
    w.r32 = -wra * (tt - a);                                     // -w (s2 - 2 Zb2)/a
    w.al3 = fma(-w.al2, w.r32, fma(-w.al1, w.r31, D3));
    return w;
}

// Left-going and right-going parts of one interface's contribution to the update (27), PAPER.md:161:
//   Gm = A^-DQ + F~  (goes to the cell on the left),  Gp = A^+DQ - F~  (goes to the cell on the right),
// with F~ of (30), limited by MC on the upwind neighbour's waves (readings A5, A6).
struct Flux3 {
    double m1, m2, m3, p1, p2, p3;
    double ft1;                         // first component of F~ alone (for the rounding order of the density update)
};

// `k`: this interface.  `u1`, `u2`, `u3`: (alpha, s, r3) of wave 1 / 2 and alpha of wave 3 at the interface that is
// upwind for that wave (k-1 if s^p_k > 0 else k+1) -- the caller selects.
__device__ __forceinline__ Flux3 interface_flux(const Waves& k, double ual1, double us1, double ur31, double ual2,
                                                double us2, double ur32, double ual3, double lam) {
    // wave 1
    const double R1 = fma(k.s1, k.s1, fma(k.r31, k.r31, 1.0));
    const double C1 = fma(us1, k.s1, fma(ur31, k.r31, 1.0));
    const double b1 = ual1 * C1 * rcp_o1(R1);
    const double as1 = fabs(k.s1);
    const double f1 = as1 * fma(-lam, as1, 1.0) * mc_half(k.al1, b1);      // (1/2)|s|(1 - lam|s|) phi alpha
    // wave 2
    const double R2 = fma(k.s2, k.s2, fma(k.r32, k.r32, 1.0));
    const double C2 = fma(us2, k.s2, fma(ur32, k.r32, 1.0));
    const double b2 = ual2 * C2 * rcp_o1(R2);
    const double as2 = fabs(k.s2);
    const double f2 = as2 * fma(-lam, as2, 1.0) * mc_half(k.al2, b2);
    // wave 3
    const double as3 = fabs(k.s3);
    const double f3 = as3 * fma(-lam, as3, 1.0) * mc_half(k.al3, ual3);
    // scalar weights of r^p in Gm / Gp
    const double g1m = fma(neg_part(k.s1), k.al1, f1), g1p = fma(pos_part(k.s1), k.al1, -f1);
    const double g2m = fma(neg_part(k.s2), k.al2, f2), g2p = fma(pos_part(k.s2), k.al2, -f2);
    const double g3m = fma(neg_part(k.s3), k.al3, f3), g3p = fma(pos_part(k.s3), k.al3, -f3);
    Flux3 F;
    F.m1 = g1m + g2m;
    F.m2 = fma(g1m, k.s1, g2m * k.s2);
    F.m3 = fma(g1m, k.r31, fma(g2m, k.r32, g3m));
    F.p1 = g1p + g2p;
    F.p2 = fma(g1p, k.s1, g2p * k.s2);
    F.p3 = fma(g1p, k.r31, fma(g2p, k.r32, g3p));
    F.ft1 = f1 + f2;
    return F;
}

// max(|s1|, |s2|) >= |s3| always (s1,2 = v +- a, a >= 0): the speed that enters M.
__device__ __forceinline__ double max_speed(const Waves& w) { return fmax(fabs(w.s1), fabs(w.s2)); }

// Inf/NaN test on the exponent bits (ALU pipe).
__device__ __forceinline__ bool not_finite(double x) { return (hi_word(x) & 0x7ff00000) == 0x7ff00000; }

}  // namespace fvnl
