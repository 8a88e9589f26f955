// fvnl_iface.cuh -- the per-interface arithmetic of the one-pass step kernels (fvnl_ws.cuh, fvnl_fused.cuh), fp64.
//
// Formulas: PAPER.md:218-245 (Roe mean of the primitive state, speeds (32)-(34), eigenvector components, alpha),
// PAPER.md:169-198 (fluctuations (28),(29), MC-limited correction (30)).  Arranged for the FP64 pipe of B200, which is
// the binding unit of this path: reciprocals and the reciprocal square root as MUFU seed + one
// third-order Newton step, the limiter without a division, min/max as compare-and-select, sign handling on the
// integer pipe.  (The three-pass comparison kernels use the separately written fvnl_math.cuh.)
#pragma once
#include "fvnl_math.cuh"

namespace fvnl {

// select by the sign bit of s: sign set -> x, else y
__device__ __forceinline__ double sel_neg(double s, double x, double y) { return hi_word(s) < 0 ? x : y; }

// compare-and-select min / max (no NaN fix-up code: a NaN anywhere ends in the output, which is checked)
__device__ __forceinline__ double dmin(double a, double b) { return b < a ? b : a; }
__device__ __forceinline__ double dmax(double a, double b) { return b > a ? b : a; }

struct Cx {       // a cell in sweep form: q2 normal, q3 transverse momentum; half primitive velocities
    double q1, q2, q3, hz2, hz3;
};
struct Wv {       // Riemann solution: W1 = al1 (1,s1,r31), W2 = al2 (1,s2,r32), W3 = (0,0,al3); v = s3
    double al1, s1, r31, al2, s2, r32, al3, v;
};
struct Fl {       // left-going (m) and right-going (p) parts of an interface's contribution to (27),
    double m1, m2, m3, p1, p2, p3;         // m = A^-DQ + F~, p = A^+DQ - F~; ft1 = first component of F~ alone
    double ft1;
};

// min_q1hi: running minimum of the high word of q1 (q1 <= 0 shows as a non-positive high word).
__device__ __forceinline__ Cx cell_of(double q1, double q2, double q3, int& min_q1hi) {
    min_q1hi = min(min_q1hi, hi_word(q1));
    Cx c;
    c.q1 = q1; c.q2 = q2; c.q3 = q3;
    const double hr = 0.5 * rcp_o1(q1);
    c.hz2 = q2 * hr;
    c.hz3 = q3 * hr;
    return c;
}

// b2 = 2(beta-1), omb2 = 1 - b2.  min_dhi tracks the sign of the square-root argument of (32),(33).
__device__ __forceinline__ Wv riemann2(const Cx& L, const Cx& R, double b2, double omb2, int& min_dhi) {
    Wv w;
    const double D1 = R.q1 - L.q1, D2 = R.q2 - L.q2, D3 = R.q3 - L.q3;
    const double Zb1 = fma(0.5, D1, L.q1);
    const double Zb2 = L.hz2 + R.hz2;
    const double Zb3 = L.hz3 + R.hz3;
    const double Phi = fma(b2, Zb1, omb2);
    const double u = rcp_o1(Zb1);
    const double v = Zb2 * u;                                    // (34)
    const double wv = Zb3 * u;
    const double tt = fma(-2.0, Zb2, v);
    const double disc = fma(v, tt, Phi);                         // (32),(33)
    min_dhi = min(min_dhi, hi_word(disc));
    const double ra = rsqrt_o1(disc);
    w.s1 = fma(disc, ra, v);                                     // v + a
    w.s2 = fma(-disc, ra, v);                                    // v - a
    w.v = v;
    const double hra = 0.5 * ra;
    w.al1 = fma(-w.s2, D1, D2) * hra;
    w.al2 = D1 - w.al1;
    const double wra = wv * ra;
    w.r31 = wra * fma(-2.0, Zb2, w.s1);                          //  w (s1 - 2 Zb2)/a
    w.r32 = wra * fma(2.0, Zb2, -w.s2);                          // -w (s2 - 2 Zb2)/a
    w.al3 = fma(-w.al2, w.r32, fma(-w.al1, w.r31, D3));
    return w;
}

// 1/(r.r) of waves 1 and 2 (denominator of theta).
__device__ __forceinline__ double rnorm(double s, double r3) { return rcp_o1(fma(s, s, fma(r3, r3, 1.0))); }

// r_K . r_k of two neighbouring interfaces (symmetric), waves 1 / 2.
__device__ __forceinline__ double rdot(double sK, double r3K, double s, double r3) { return fma(sK, s, fma(r3K, r3, 1.0)); }

// Half of phi(b/a) a for the MC limiter phi(theta) = max(0, min((1+theta)/2, 2, 2 theta)):
//   phi(b/a) a = 2 sgn(a) max(0, min((|a| + B)/4, |a|, B)),  B = sgn(a) b.      a = 0 gives 0 (reading A5).
__device__ __forceinline__ double mc_half2(double a, double b) {
    const double A = fabs(a);
    const double B = xor_sign(b, a);
    const double q = 0.25 * (A + B);
    const double m = dmin(dmin(A, B), q);
    const double r = sel_neg(m, 0.0, m);
    return xor_sign(r, a);
}

// k: the interface; b_p = alpha_K^p (r_K.r_k)/(r_k.r_k) of the upwind interface K (b3 = alpha_K^3).  (28)-(30).
__device__ __forceinline__ Fl flux2(const Wv& k, double b1, double b2, double b3, double lam) {
    const double a1 = fabs(k.s1), a2 = fabs(k.s2), a3 = fabs(k.v);
    const double f1 = a1 * fma(-lam, a1, 1.0) * mc_half2(k.al1, b1);
    const double f2 = a2 * fma(-lam, a2, 1.0) * mc_half2(k.al2, b2);
    const double f3 = a3 * fma(-lam, a3, 1.0) * mc_half2(k.al3, b3);
    const double g1m = fma(neg_part(k.s1), k.al1, f1), g1p = fma(k.s1, k.al1, -g1m);
    const double g2m = fma(neg_part(k.s2), k.al2, f2), g2p = fma(k.s2, k.al2, -g2m);
    const double g3m = fma(neg_part(k.v), k.al3, f3), g3p = fma(k.v, k.al3, -g3m);
    Fl F;
    F.m1 = g1m + g2m;
    F.m2 = fma(g1m, k.s1, g2m * k.s2);
    F.m3 = fma(g1m, k.r31, fma(g2m, k.r32, g3m));
    F.p1 = g1p + g2p;
    F.p2 = fma(g1p, k.s1, g2p * k.s2);
    F.p3 = fma(g1p, k.r31, fma(g2p, k.r32, g3p));
    F.ft1 = f1 + f2;
    return F;
}

// The density component of the update (27).  q1 is of order one while its increment is of order of the perturbation, so
// the two roundings of  (q - lam (A+DQ_l + A-DQ_r)) - lam (F~_r - F~_l)  (evaluated in this order) are the
// largest round-off of a step by orders of magnitude, and a random walk of one-ulp differences over hundreds of steps
// and 10^6..10^8 cells would by itself exceed the 1e-10 parity bar.  The CUDA path therefore rounds where the definition
// rounds: two separate, uncontracted subtractions.  sum = p1_l + m1_r (both halves as produced by flux2), ft_l, ft_r =
// first component of F~ at the two interfaces.
__device__ __forceinline__ double update_q1(double q, double lam, double sum, double ft_l, double ft_r) {
    const double s2 = __dsub_rn(ft_r, ft_l);                      // F~_r - F~_l
    const double s1 = __dsub_rn(sum, s2);                         // A+DQ_l + A-DQ_r
    const double u = __dsub_rn(q, __dmul_rn(lam, s1));
    return __dsub_rn(u, __dmul_rn(lam, s2));
}

}  // namespace fvnl
