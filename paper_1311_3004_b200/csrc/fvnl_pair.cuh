// fvnl_pair.cuh -- the per-interface arithmetic of the fused kernels, written once for a scalar (double) and for a
// PAIR of independent problems (V2).
//
// Why pairs.  A warp issues in order, and a dependent FP64 operation waits 9 cycles for its operand (measured on
// B200).  The Riemann solve is one long dependency chain (two Newton-refined MUFU seeds in sequence), and ptxas keeps
// independent chains in the order the source gives them; with the x-sweep's and the y-sweep's Riemann solves (or
// limited fluxes) written one after the other the FP64 pipe idles most of the time.  Evaluating the x-problem and the
// y-problem as the two lanes of a V2 puts two independent instructions next to each other at every step of the chain.
// Formulas: PAPER.md:218-245 (Roe mean, speeds (32)-(34), eigenvector components, alpha)
// (fluctuations (28),(29), MC-limited correction (30)); same arrangement as fvnl_math.cuh.
#pragma once
#include <type_traits>
#include "fvnl_math.cuh"

namespace fvnl {

using ::fabs;
using ::fma;

struct V2 { double a, b; };
struct I2 { int a, b; };

template <class T> struct is_v2 : std::false_type {};
template <> struct is_v2<V2> : std::true_type {};
template <class... Ts> constexpr bool any_v2 = (is_v2<Ts>::value || ...);

__device__ __forceinline__ double e0(double x) { return x; }
__device__ __forceinline__ double e1(double x) { return x; }
__device__ __forceinline__ double e0(V2 x) { return x.a; }
__device__ __forceinline__ double e1(V2 x) { return x.b; }

// elementwise operators for any mix of V2 and double with at least one V2
template <class A, class B, std::enable_if_t<any_v2<A, B>, int> = 0>
__device__ __forceinline__ V2 operator+(A x, B y) { return V2{e0(x) + e0(y), e1(x) + e1(y)}; }
template <class A, class B, std::enable_if_t<any_v2<A, B>, int> = 0>
__device__ __forceinline__ V2 operator-(A x, B y) { return V2{e0(x) - e0(y), e1(x) - e1(y)}; }
template <class A, class B, std::enable_if_t<any_v2<A, B>, int> = 0>
__device__ __forceinline__ V2 operator*(A x, B y) { return V2{e0(x) * e0(y), e1(x) * e1(y)}; }
__device__ __forceinline__ V2 operator-(V2 x) { return V2{-x.a, -x.b}; }
template <class A, class B, class C, std::enable_if_t<any_v2<A, B, C>, int> = 0>
__device__ __forceinline__ V2 fma(A x, B y, C z) { return V2{::fma(e0(x), e0(y), e0(z)), ::fma(e1(x), e1(y), e1(z))}; }
__device__ __forceinline__ V2 fabs(V2 x) { return V2{::fabs(x.a), ::fabs(x.b)}; }

// the scalar helpers of fvnl_math.cuh, elementwise
__device__ __forceinline__ I2 hi_word(V2 x) { return I2{hi_word(x.a), hi_word(x.b)}; }
__device__ __forceinline__ V2 rcp_o1(V2 x) {                              // seeds first, then the two Newton chains in step
    double ya, yb;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(ya) : "d"(x.a));
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(yb) : "d"(x.b));
    const double ea = ::fma(-x.a, ya, 1.0), eb = ::fma(-x.b, yb, 1.0);
    const double ta = ::fma(ea, ea, ea), tb = ::fma(eb, eb, eb);
    return V2{::fma(ya, ta, ya), ::fma(yb, tb, yb)};
}
__device__ __forceinline__ V2 rsqrt_o1(V2 x) {
    double ya, yb;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(ya) : "d"(x.a));
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(yb) : "d"(x.b));
    const double ta = x.a * ya, tb = x.b * yb;
    const double ea = ::fma(-ta, ya, 1.0), eb = ::fma(-tb, yb, 1.0);
    const double pa = ::fma(0.375, ea, 0.5), pb = ::fma(0.375, eb, 0.5);
    const double qa = ea * pa, qb = eb * pb;
    return V2{::fma(ya, qa, ya), ::fma(yb, qb, yb)};
}
__device__ __forceinline__ V2 xor_sign(V2 x, V2 s) { return V2{xor_sign(x.a, s.a), xor_sign(x.b, s.b)}; }
__device__ __forceinline__ V2 neg_part(V2 s) { return V2{neg_part(s.a), neg_part(s.b)}; }

// select by the sign bit of s: sign set -> x, else y
__device__ __forceinline__ double sel_neg(double s, double x, double y) { return hi_word(s) < 0 ? x : y; }
__device__ __forceinline__ V2 sel_neg(V2 s, V2 x, V2 y) { return V2{sel_neg(s.a, x.a, y.a), sel_neg(s.b, x.b, y.b)}; }

__device__ __forceinline__ double zero_like(double) { return 0.0; }
__device__ __forceinline__ V2 zero_like(V2) { return V2{0.0, 0.0}; }

// compare-and-select min / max (no NaN fix-up code: a NaN anywhere ends in the output, which is checked)
__device__ __forceinline__ double dmin(double a, double b) { return b < a ? b : a; }
__device__ __forceinline__ double dmax(double a, double b) { return b > a ? b : a; }
__device__ __forceinline__ V2 dmin(V2 x, V2 y) { return V2{dmin(x.a, y.a), dmin(x.b, y.b)}; }

// running minimum of high words (sign tracking for the flags)
__device__ __forceinline__ void track_min(int& acc, double x) { acc = min(acc, hi_word(x)); }
__device__ __forceinline__ void track_min(I2& acc, V2 x) { acc.a = min(acc.a, hi_word(x.a)); acc.b = min(acc.b, hi_word(x.b)); }
template <class T> struct hi_of { using type = int; };
template <> struct hi_of<V2> { using type = I2; };

// ---- cells, Riemann solves, limited fluxes; T = double or V2 ------------------------------------------------------
template <class T> struct CxT {       // a cell in sweep form: q2 normal, q3 transverse momentum; half primitive velocities
    T q1, q2, q3, hz2, hz3;
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

template <class T>
__device__ __forceinline__ CxT<T> cell_of(T q1, T q2, T q3, typename hi_of<T>::type& min_q1hi) {
    track_min(min_q1hi, q1);                                     // q1 <= 0 shows as a non-positive high word
    CxT<T> c;
    c.q1 = q1; c.q2 = q2; c.q3 = q3;
    const T hr = 0.5 * rcp_o1(q1);
    c.hz2 = q2 * hr;
    c.hz3 = q3 * hr;
    return c;
}

// b2 = 2(beta-1), omb2 = 1 - b2.  min_dhi tracks the sign of the square-root argument of (32),(33).
template <class T>
__device__ __forceinline__ WvT<T> riemann2(const CxT<T>& L, const CxT<T>& R, double b2, double omb2,
                                           typename hi_of<T>::type& min_dhi) {
    WvT<T> w;
    const T D1 = R.q1 - L.q1, D2 = R.q2 - L.q2, D3 = R.q3 - L.q3;
    const T Zb1 = fma(0.5, D1, L.q1);
    const T Zb2 = L.hz2 + R.hz2;
    const T Zb3 = L.hz3 + R.hz3;
    const T Phi = fma(b2, Zb1, omb2);
    const T u = rcp_o1(Zb1);
    const T v = Zb2 * u;                                         // (34)
    const T wv = Zb3 * u;
    const T tt = fma(-2.0, Zb2, v);
    const T disc = fma(v, tt, Phi);                              // (32),(33)
    track_min(min_dhi, disc);
    const T ra = rsqrt_o1(disc);
    w.s1 = fma(disc, ra, v);                                     // v + a
    w.s2 = fma(-disc, ra, v);                                    // v - a
    w.v = v;
    const T hra = 0.5 * ra;
    w.al1 = fma(-w.s2, D1, D2) * hra;
    w.al2 = D1 - w.al1;
    const T wra = wv * ra;
    w.r31 = wra * fma(-2.0, Zb2, w.s1);                          //  w (s1 - 2 Zb2)/a
    w.r32 = wra * fma(2.0, Zb2, -w.s2);                          // -w (s2 - 2 Zb2)/a
    w.al3 = fma(-w.al2, w.r32, fma(-w.al1, w.r31, D3));
    return w;
}

// 1/(r.r) of waves 1 and 2 (denominator of theta).
template <class T> __device__ __forceinline__ T rnorm(T s, T r3) { return rcp_o1(fma(s, s, fma(r3, r3, 1.0))); }

// r_K . r_k of two neighbouring interfaces (symmetric), waves 1 / 2.
template <class T> __device__ __forceinline__ T rdot(T sK, T r3K, T s, T r3) { return fma(sK, s, fma(r3K, r3, 1.0)); }

// Half of phi(b/a) a, MC limiter, as mc_half of fvnl_math.cuh.
template <class T> __device__ __forceinline__ T mc_half2(T a, T b) {
    const T A = fabs(a);
    const T B = xor_sign(b, a);
    const T q = 0.25 * (A + B);
    const T m = dmin(dmin(A, B), q);
    const T r = sel_neg(m, zero_like(m), m);
    return xor_sign(r, a);
}

// k: the interface; b_p = alpha_K^p (r_K.r_k)/(r_k.r_k) of the upwind interface K (b3 = alpha_K^3).  (28)-(30).
template <class T, class LAM>
__device__ __forceinline__ FlT<T> flux2(const WvT<T>& k, T b1, T b2, T b3, LAM lam) {
    const T a1 = fabs(k.s1), a2 = fabs(k.s2), a3 = fabs(k.v);
    const T f1 = a1 * fma(-lam, a1, 1.0) * mc_half2(k.al1, b1);
    const T f2 = a2 * fma(-lam, a2, 1.0) * mc_half2(k.al2, b2);
    const T f3 = a3 * fma(-lam, a3, 1.0) * mc_half2(k.al3, b3);
    const T g1m = fma(neg_part(k.s1), k.al1, f1), g1p = fma(k.s1, k.al1, -g1m);
    const T g2m = fma(neg_part(k.s2), k.al2, f2), g2p = fma(k.s2, k.al2, -g2m);
    const T g3m = fma(neg_part(k.v), k.al3, f3), g3p = fma(k.v, k.al3, -g3m);
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

// ---- packing two scalar problems into the lanes of a pair and back ------------------------------------------------
__device__ __forceinline__ V2 pk(double a, double b) { return V2{a, b}; }
__device__ __forceinline__ CxT<V2> pk(const Cx& a, const Cx& b) {
    return CxT<V2>{pk(a.q1, b.q1), pk(a.q2, b.q2), pk(a.q3, b.q3), pk(a.hz2, b.hz2), pk(a.hz3, b.hz3)};
}
__device__ __forceinline__ WvT<V2> pk(const Wv& a, const Wv& b) {
    return WvT<V2>{pk(a.al1, b.al1), pk(a.s1, b.s1), pk(a.r31, b.r31), pk(a.al2, b.al2),
                   pk(a.s2, b.s2), pk(a.r32, b.r32), pk(a.al3, b.al3), pk(a.v, b.v)};
}
__device__ __forceinline__ Cx lane_a(const CxT<V2>& c) { return Cx{c.q1.a, c.q2.a, c.q3.a, c.hz2.a, c.hz3.a}; }
__device__ __forceinline__ Cx lane_b(const CxT<V2>& c) { return Cx{c.q1.b, c.q2.b, c.q3.b, c.hz2.b, c.hz3.b}; }
__device__ __forceinline__ Wv lane_a(const WvT<V2>& w) { return Wv{w.al1.a, w.s1.a, w.r31.a, w.al2.a, w.s2.a, w.r32.a, w.al3.a, w.v.a}; }
__device__ __forceinline__ Wv lane_b(const WvT<V2>& w) { return Wv{w.al1.b, w.s1.b, w.r31.b, w.al2.b, w.s2.b, w.r32.b, w.al3.b, w.v.b}; }
__device__ __forceinline__ Fl lane_a(const FlT<V2>& f) { return Fl{f.m1.a, f.m2.a, f.m3.a, f.p1.a, f.p2.a, f.p3.a, f.ft1.a}; }
__device__ __forceinline__ Fl lane_b(const FlT<V2>& f) { return Fl{f.m1.b, f.m2.b, f.m3.b, f.p1.b, f.p2.b, f.p3.b, f.ft1.b}; }

}  // namespace fvnl
