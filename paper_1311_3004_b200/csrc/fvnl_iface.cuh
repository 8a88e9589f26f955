// fvnl_iface.cuh -- the per-interface arithmetic of the one-pass step kernels (fvnl_ws.cuh, fvnl_fused.cuh), written
// once for the two precisions of the library: T = double (the paper's) and T = float.
//
// Formulas: PAPER.md:218-245 (Roe mean of the primitive state, speeds (32)-(34), eigenvector components, alpha),
// PAPER.md:169-198 (fluctuations (28),(29), MC-limited correction (30)).
//
// fp64: arranged for the FP64 pipe of B200, the binding unit of that path: reciprocals and the
// reciprocal square root as MUFU seed + one third-order Newton step, the limiter without a division, min/max as
// compare-and-select, sign handling on the integer pipe.
//
// fp32: PERTURBATION FORM.  The density variable of a cell is rho' = q1 - 1, not q1: differences of neighbouring cells, the
// Roe mean Zbar1 - 1, Phi - 1 and the update (27) are formed from rho' directly, so that fp32 round-off is relative to the
// perturbation (1e-6 .. 1e-3) and not to the unit background (one ulp of 1.0f is 1e-4 .. 1e-1 of it).  Reciprocals and
// square roots are the MUFU approximations (1-2 ulp of fp32), min/max are FMNMX.
// (The three-pass comparison kernels use the separately written fvnl_math.cuh.)
#pragma once
#include "fvnl_math.cuh"

namespace fvnl {

// ---- what differs between the two precisions -------------------------------------------------------------------
template <class T> struct Num;

template <> struct Num<double> {
    using T2 = double2;
    static constexpr bool perturbation = false;               // density variable of a cell: q1 itself
    static constexpr int inf_hi = 0x7ff00000;                 // |hi word| >= this: Inf / NaN
    __device__ static __forceinline__ int hi(double x) { return __double2hiint(x); }       // word with sign and exponent
    __device__ static __forceinline__ double rcp(double x) { return rcp_o1(x); }
    __device__ static __forceinline__ double rsqrt(double x) { return rsqrt_o1(x); }
    __device__ static __forceinline__ double xor_sign(double x, double s) { return fvnl::xor_sign(x, s); }
    __device__ static __forceinline__ double neg_part(double s) { return hi(s) < 0 ? s : 0.0; }
    __device__ static __forceinline__ double min2(double a, double b) { return b < a ? b : a; }   // compare-and-select:
    __device__ static __forceinline__ double max2(double a, double b) { return b > a ? b : a; }   // no NaN fix-up code
    __device__ static __forceinline__ double relu(double m) { return hi(m) < 0 ? 0.0 : m; }
    __device__ static __forceinline__ double2 make2(double a, double b) { return make_double2(a, b); }
};

template <> struct Num<float> {
    using T2 = float2;
    static constexpr bool perturbation = true;                // density variable of a cell: rho' = q1 - 1
    static constexpr int inf_hi = 0x7f800000;
    __device__ static __forceinline__ int hi(float x) { return __float_as_int(x); }
    __device__ static __forceinline__ float rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
    __device__ static __forceinline__ float rsqrt(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
    __device__ static __forceinline__ float xor_sign(float x, float s) {
        return __int_as_float(__float_as_int(x) ^ (__float_as_int(s) & 0x80000000));
    }
    __device__ static __forceinline__ float neg_part(float s) { return fminf(s, 0.0f); }
    __device__ static __forceinline__ float min2(float a, float b) { return fminf(a, b); }
    __device__ static __forceinline__ float max2(float a, float b) { return fmaxf(a, b); }
    __device__ static __forceinline__ float relu(float m) { return fmaxf(m, 0.0f); }
    __device__ static __forceinline__ float2 make2(float a, float b) { return make_float2(a, b); }
};

// select by the sign bit of s: sign set -> x, else y
template <class T> __device__ __forceinline__ T sel_neg(T s, T x, T y) { return Num<T>::hi(s) < 0 ? x : y; }
__device__ __forceinline__ double dmin(double a, double b) { return Num<double>::min2(a, b); }
__device__ __forceinline__ double dmax(double a, double b) { return Num<double>::max2(a, b); }

template <class T> struct CxT {       // a cell in sweep form: q1 = density variable (q1, or rho' in fp32), q2 normal and q3
    T q1, q2, q3, hz2, hz3;           // transverse momentum; half primitive velocities
};
template <class T> struct WvT {       // Riemann solution: W1 = al1 (1,s1,r31), W2 = al2 (1,s2,r32), W3 = (0,0,al3); v = s3
    T al1, s1, r31, al2, s2, r32, al3, v;
};
template <class T> struct FlT {       // left-going (m) and right-going (p) parts of an interface's contribution to (27),
    T m1, m2, m3, p1, p2, p3;         // m = A^-DQ + F~, p = A^+DQ - F~; ft1 = first component of F~ alone
    T ft1;
};
using Cx = CxT<double>;
using Wv = WvT<double>;
using Fl = FlT<double>;

// min_q1hi: running minimum of the sign/exponent word of the density (q1 <= 0 shows as a non-positive word).
template <class T>
__device__ __forceinline__ CxT<T> cell_of(T q1, T q2, T q3, int& min_q1hi) {
    const T dens = Num<T>::perturbation ? T(1) + q1 : q1;
    min_q1hi = min(min_q1hi, Num<T>::hi(dens));
    CxT<T> c;
    c.q1 = q1; c.q2 = q2; c.q3 = q3;
    const T hr = T(0.5) * Num<T>::rcp(dens);
    c.hz2 = q2 * hr;
    c.hz3 = q3 * hr;
    return c;
}

// b2 = 2(beta-1), omb2 = 1 - b2.  min_dhi tracks the sign of the square-root argument of (32),(33).
template <class T>
__device__ __forceinline__ WvT<T> riemann2(const CxT<T>& L, const CxT<T>& R, T b2, T omb2, int& min_dhi) {
    WvT<T> w;
    const T D1 = R.q1 - L.q1, D2 = R.q2 - L.q2, D3 = R.q3 - L.q3;
    T Zb1, Phi;
    if (Num<T>::perturbation) {
        const T h = T(0.5) * (L.q1 + R.q1);                      // Zbar1 - 1
        Zb1 = T(1) + h;
        Phi = fma(b2, h, T(1));
    } else {
        Zb1 = fma(T(0.5), D1, L.q1);
        Phi = fma(b2, Zb1, omb2);
    }
    const T Zb2 = L.hz2 + R.hz2;
    const T Zb3 = L.hz3 + R.hz3;
    const T u = Num<T>::rcp(Zb1);
    const T v = Zb2 * u;                                         // (34)
    const T wv = Zb3 * u;
    const T tt = fma(T(-2), Zb2, v);
    const T disc = fma(v, tt, Phi);                              // (32),(33)
    min_dhi = min(min_dhi, Num<T>::hi(disc));
    const T ra = Num<T>::rsqrt(disc);
    w.s1 = fma(disc, ra, v);                                     // v + a
    w.s2 = fma(-disc, ra, v);                                    // v - a
    w.v = v;
    const T hra = T(0.5) * ra;
    w.al1 = fma(-w.s2, D1, D2) * hra;
    w.al2 = D1 - w.al1;
    const T wt = wv * ra * tt;                                   // s1 - 2 Zb2 = tt + a, s2 - 2 Zb2 = tt - a, and a/a = 1:
    w.r31 = wv + wt;                                             //  w (s1 - 2 Zb2)/a = w + w tt/a
    w.r32 = wv - wt;                                             // -w (s2 - 2 Zb2)/a = w - w tt/a
    w.al3 = fma(-w.al2, w.r32, fma(-w.al1, w.r31, D3));
    return w;
}

// 1/(r.r) of waves 1 and 2 (denominator of theta).
template <class T> __device__ __forceinline__ T rnorm(T s, T r3) { return Num<T>::rcp(fma(s, s, fma(r3, r3, T(1)))); }

// r_K . r_k of two neighbouring interfaces (symmetric), waves 1 / 2.
template <class T> __device__ __forceinline__ T rdot(T sK, T r3K, T s, T r3) { return fma(sK, s, fma(r3K, r3, T(1))); }

// Half of phi(b/a) a for the MC limiter phi(theta) = max(0, min((1+theta)/2, 2, 2 theta)):
//   phi(b/a) a = 2 sgn(a) max(0, min((|a| + B)/4, |a|, B)),  B = sgn(a) b.      a = 0 gives 0 (reading A5).
template <class T> __device__ __forceinline__ T mc_half2(T a, T b) {
    const T A = fabs(a);
    const T B = Num<T>::xor_sign(b, a);
    const T q = T(0.25) * (A + B);
    const T m = Num<T>::min2(Num<T>::min2(A, B), q);
    return Num<T>::xor_sign(Num<T>::relu(m), a);
}

// k: the interface; b_p = alpha_K^p (r_K.r_k)/(r_k.r_k) of the upwind interface K (b3 = alpha_K^3).  (28)-(30).
template <class T>
__device__ __forceinline__ FlT<T> flux2(const WvT<T>& k, T b1, T b2, T b3, T lam) {
    const T a1 = fabs(k.s1), a2 = fabs(k.s2), a3 = fabs(k.v);
    // |s| (1 - lam |s|) as |s| - (lam |s|) |s|: no immediate operand next to lam, which then stays in a uniform register
    const T f1 = fma(-(lam * a1), a1, a1) * mc_half2(k.al1, b1);
    const T f2 = fma(-(lam * a2), a2, a2) * mc_half2(k.al2, b2);
    const T f3 = fma(-(lam * a3), a3, a3) * mc_half2(k.al3, b3);
    const T g1m = fma(Num<T>::neg_part(k.s1), k.al1, f1), g1p = fma(k.s1, k.al1, -g1m);
    const T g2m = fma(Num<T>::neg_part(k.s2), k.al2, f2), g2p = fma(k.s2, k.al2, -g2m);
    const T g3m = fma(Num<T>::neg_part(k.v), k.al3, f3), g3p = fma(k.v, k.al3, -g3m);
    FlT<T> F;
    F.m1 = g1m + g2m;
    F.m2 = fma(g1m, k.s1, g2m * k.s2);
    F.m3 = fma(g1m, k.r31, fma(g2m, k.r32, g3m));
    F.p1 = g1p + g2p;
    F.p2 = fma(g1p, k.s1, g2p * k.s2);
    F.p3 = fma(g1p, k.r31, fma(g2p, k.r32, g3p));
    F.ft1 = f1 + f2;
    return F;
}

// The density component of the update (27).  fp64: q1 is of order one while its increment is of order of the perturbation,
// so the two roundings of  (q - lam (A+DQ_l + A-DQ_r)) - lam (F~_r - F~_l)  (evaluated in this order) are the
// largest round-off of a step by orders of magnitude, and a random walk of one-ulp differences over hundreds of steps
// and 10^6..10^8 cells would by itself exceed the 1e-10 parity bar.  The fp64 path therefore rounds where the definition
// rounds: two separate, uncontracted subtractions.  sum = p1_l + m1_r (both halves as produced by flux2), ft_l, ft_r =
// first component of F~ at the two interfaces.
__device__ __forceinline__ double update_q1(double q, double lam, double sum, double ft_l, double ft_r) {
    const double s2 = __dsub_rn(ft_r, ft_l);                      // F~_r - F~_l
    const double s1 = __dsub_rn(sum, s2);                         // A+DQ_l + A-DQ_r
    const double u = __dsub_rn(q, __dmul_rn(lam, s1));
    return __dsub_rn(u, __dmul_rn(lam, s2));
}
// fp32: the density variable is the perturbation itself, its round-off is relative to the perturbation: one FMA.
__device__ __forceinline__ float update_q1(float rho, float lam, float sum, float, float) { return fmaf(-lam, sum, rho); }

}  // namespace fvnl
