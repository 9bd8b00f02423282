// device_math.cuh -- per-cell and per-interface arithmetic of the hot path (sm_100a).
//
// Everything here is the CUDA side's own restatement of DESIGN.md section 2 (steps a2..a7'); it shares
// no source with oracle/.  The formulas are algebraically those of the paper's schemes (WENO5/7 on
// LLF-split fluxes; MUSTA-FORCE with MUSCL/minmod) but arranged for the
// fp64 pipe: undivided differences, fused multiply-adds, cross-multiplied nonlinear weights and one
// reciprocal per pair of reconstructions.  The rearrangements change rounding only.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#define HD __host__ __device__ __forceinline__

namespace hydro {

enum { NF = 5 };                       // E, Mx, My, Mz, R
// primitive arrays kept beside a state: v_x, v_y, v_z, p, a_x, a_y, a_z (a2-a3 of every cell, made once per stage)
enum { W_V = 0, W_P = 3, W_AX = 4 };
enum { NW = 7 };

template <class T> HD T tfma(T a, T b, T c);
template <> HD double tfma<double>(double a, double b, double c) { return fma(a, b, c); }
template <> HD float tfma<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <class T> HD T tsqrt(T x);
template <> HD double tsqrt<double>(double x) { return sqrt(x); }
template <> HD float tsqrt<float>(float x) { return sqrtf(x); }
template <class T> HD T tabs(T x);   // |x| as an operand modifier, not a compare and two selects
template <> HD double tabs<double>(double x) { return fabs(x); }
template <> HD float tabs<float>(float x) { return fabsf(x); }
template <class T> HD T tmax(T a, T b);
template <> HD double tmax<double>(double a, double b) { return fmax(a, b); }
template <> HD float tmax<float>(float a, float b) { return fmaxf(a, b); }
// max of two NON-NEGATIVE numbers.  fp64 on the device: non-negative doubles order like their bit patterns, so
// the compare runs in the integer pipe instead of occupying the fp64 pipe (DSETP + selects)
template <class T> HD T max_nonneg(T a, T b) { return tmax(a, b); }
#ifdef __CUDA_ARCH__
template <>
__device__ __forceinline__ double max_nonneg<double>(double a, double b) {
    return __longlong_as_double(max(__double_as_longlong(a), __double_as_longlong(b)));
}
#endif
template <class T> HD T tmin(T a, T b);
template <> HD double tmin<double>(double a, double b) { return fmin(a, b); }
template <> HD float tmin<float>(float a, float b) { return fminf(a, b); }

// Reciprocal of a positive, finite, normal number.  fp64: MUFU.RCP64H seed plus one cubically convergent
// step = 3 DFMA, error about 1 ulp, no special-case path.  fp32: the hardware reciprocal.
HD double fast_rcp(double x) {
#ifdef __CUDA_ARCH__
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    // one cubically convergent step: y (1 + e + e^2), e = 1 - x y.  The seed is good to about 2^-20, so the
    // result to about 2^-60 before rounding; three dependent instructions instead of the four of two Newton steps
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
#else
    return 1.0 / x;
#endif
}
HD float fast_rcp(float x) {
#ifdef __CUDA_ARCH__
    float y;   // MUFU.RCP alone: 1 ulp-level, against the correctly rounded __frcp_rn's fix-up sequence
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
#else
    return 1.0f / x;
#endif
}

// Square root of a positive, finite, normal number.  fp64: MUFU.RSQ64H seed y (relative error below 2^-20) plus ONE
// cubically convergent step on s = x y: with e = 1 - s y = 1 - x y^2 the root is s (1 - e)^(-1/2) =
// s (1 + e/2 + 3 e^2/8 + O(e^3)), remainder below 2^-58; 5 fp64-pipe instructions, error about 1 ulp, no special-case
// path.  fp32: the hardware square root.
HD double fast_sqrt(double x) {
#ifdef __CUDA_ARCH__
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double s = x * y;
    const double e = fma(-s, y, 1.0);
    const double pe = fma(0.375, e, 0.5) * e;
    return fma(s, pe, s);
#else
    return sqrt(x);
#endif
}
HD float fast_sqrt(float x) {
#ifdef __CUDA_ARCH__
    float y;   // MUFU.SQRT alone
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
#else
    return sqrtf(x);
#endif
}

// ------------------------------------------------------------------------------------------------
// a2. conserved -> primitive, closed form for p = e/3 (a2; reading Q16).
//   s = sqrt(4E^2 - 3M^2);  v_i = 3 M_i/(2E + s);  e = 3(E^2 - M^2)/(s + E);  p = e/3.
// Returns winv = 3/(2E+s) (so that v_i = M_i * winv) and p.  The clamp E >= 1e-300,
// |M| <= (1-1e-12) E raises flag; the caller's E and M are left alone (the physical flux keeps using
// them), the rescaling of M goes into winv.
template <class T>
HD bool below_floor(T E) {   // true for NaN and +Inf too: a non-finite energy must raise the flag (reading Q16)
    return !(E >= (T)1e-300) || E > (T)(sizeof(T) == 8 ? 1.7976931348623157e308 : 3.4028234e38);
}
#ifdef __CUDA_ARCH__
// fp64: positive doubles order like their bit patterns, so the floor test is an integer compare on the high
// word (negative E fails it through the sign bit); keeps one compare off the fp64 pipe
template <>
__device__ __forceinline__ bool below_floor<double>(double E) {
    // high word of 1e-300 = 0x01a56e1fc2f8f359; 0x7ff00000 and above is +Inf / +NaN: one unsigned compare of
    // (hi - floor) against the width of the admissible band rejects negative, tiny, infinite and NaN energies
    return (unsigned)(__double2hiint(E) - 0x01a56e1f) >= (unsigned)(0x7ff00000 - 0x01a56e1f);
}
#endif

template <class T>
HD void con2prim(T E, T M0, T M1, T M2, T& winv, T& p, T& v2, int& flag) {
    if (below_floor(E)) {
        E = (T)1e-300;
        flag = 1;
    }
    T m2 = tfma(M0, M0, tfma(M1, M1, M2 * M2));
    T t = E * E;
    T sc = (T)1;
    const T c2 = ((T)1 - (T)1e-12) * ((T)1 - (T)1e-12);
    if (!(m2 <= c2 * t)) {   // |M| > (1 - 1e-12) E up to rounding, or NaN: settle it with the square root (rare path)
        const T lim = ((T)1 - (T)1e-12) * E;
        const T mabs = tsqrt(m2);
        if (!(mabs <= lim)) {   // a NaN momentum lands here as well: flagged
            sc = lim / mabs;
            m2 = lim * lim;
            flag = 1;
        }
    }
    // one reciprocal serves both quotients: 1/((2E+s)(s+E))
    const T s = fast_sqrt(tfma((T)4, t, (T)-3 * m2));
    const T d1 = tfma((T)2, E, s), d2 = s + E;
    const T r = fast_rcp(d1 * d2);
    const T w = (T)3 * (r * d2);
    p = (t - m2) * (r * d1);
    v2 = m2 * w * w;
    winv = w * sc;
}

// The constant-pressure closure p = p0 (reading Q14): v_i = M_i/(E + p0), p = p0; same outputs
// and clamp policy (E + p0 >= 1e-300, |M| <= (1 - 1e-12)(E + p0)) as con2prim.
template <class T>
HD void con2prim_p0(T E, T M0, T M1, T M2, T p0, T& winv, T& p, T& v2, int& flag) {
    T H = E + p0;
    if (!(H >= (T)1e-300)) {
        H = (T)1e-300;
        flag = 1;
    }
    T m2 = tfma(M0, M0, tfma(M1, M1, M2 * M2));
    const T lim = ((T)1 - (T)1e-12) * H;
    T sc = (T)1;
    if (!(m2 <= lim * lim)) {
        const T mabs = tsqrt(m2);
        if (!(mabs <= lim)) {
            sc = lim / mabs;
            m2 = lim * lim;
            flag = 1;
        }
    }
    const T w = fast_rcp(H);
    p = p0;
    v2 = m2 * w * w;
    winv = w * sc;
}

// Equation of state of a context.  kind 0: p = e/3 (reading Q2); 1: p = p0 (reading Q14);
// 2: tabulated barotropic p(e) (second half of N1): n values on the uniform grid e_min + i de in the caller's DEVICE
// memory (always doubles), interpolated linearly, the end segments continued; c_s^2 = dp/de is the segment's slope.
struct EosArgs {
    int kind;
    double p0;
    const double* tab;
    int n;
    double e_min, de;
};

// con2prim for the tabulated closure (N1).  p(e) is piecewise linear on the knots e_k = e_min + k de, first and last
// segment continued.  The energy density is the root of
//     g(e) = (E - e)(E + p(e)) - M^2,
// which has the sign of E - M^2/(E + p(e)) - e wherever E + p > 0 and, like it, falls through its single root.  On
// segment k, with x = e - e_k, H_k = E + p_k, D_k = E - e_k and slope c (= c_s^2 of the segment),
//     g = -c x^2 - B x + g_k,   B = H_k - c D_k = (1 - c) E + p_k + c e_k > 0,   g_k = D_k H_k - M^2 = g(e_k),
// so the root of the segment's parabola is x = 2 g_k / (B + sqrt(B^2 + 4 c g_k)) in closed form: no iteration on e.
// What is searched is the segment.  x < 0 says g_k < 0, the root lies below e_k; x >= de says g(e_{k+1}) >= 0, it
// lies at or above e_{k+1}; either way the bracket [lo, hi] of candidate segments shrinks, and the next candidate is
// the segment the extrapolated root e_k + x points to (on a smooth table that is the right one or its neighbour),
// plain bisection of the bracket after 8 such jumps.  At most 8 + log2(n) candidates, typically one or two.
// All in double whatever T is.  Same outputs and clamp policy (E >= 1e-300, |M| <= (1 - 1e-12) E, reading Q16) as
// con2prim, plus cs2.  A root within rounding of a knot may take the slope of either neighbour segment.
template <class T>
HD void con2prim_tab(T E_, T M0, T M1, T M2, const EosArgs& eos, T& winv, T& p, T& v2, T& cs2, int& flag) {
    double E = (double)E_;
    if (below_floor(E_)) {
        E = 1e-300;
        flag = 1;
    }
    double m2 = (double)M0 * M0 + (double)M1 * M1 + (double)M2 * M2;
    double sc = 1.0;
    const double lim = (1.0 - 1e-12) * E;
    if (!(m2 <= lim * lim)) {
        const double mabs = sqrt(m2);
        if (!(mabs <= lim)) {   // NaN momentum lands here too
            sc = lim / mabs;
            m2 = lim * lim;
            flag = 1;
        }
    }
    const double de = eos.de, inv_de = 1.0 / de;
    int lo = 0, hi = eos.n - 2;
    double t = (E - eos.e_min) * inv_de;   // first candidate: the segment of e = E (the root is at or below E)
    double pk = 0.0, c = 0.0, x = 0.0;
    for (int it = 0; it < 96; ++it) {
        const int k = t >= (double)hi ? hi : (t > (double)lo ? (int)t : lo);   // a NaN picks lo
#ifdef __CUDA_ARCH__
        pk = __ldg(eos.tab + k);
        const double pn = __ldg(eos.tab + k + 1);
#else
        pk = eos.tab[k];
        const double pn = eos.tab[k + 1];
#endif
        const double ek = fma((double)k, de, eos.e_min);
        c = (pn - pk) * inv_de;
        const double Hk = E + pk, Dk = E - ek;
        const double gk = fma(Dk, Hk, -m2);
        const double B = fma(-c, Dk, Hk);
        const double disc = fma(B, B, 4.0 * c * gk);
        x = 2.0 * gk / (B + sqrt(disc > 0.0 ? disc : 0.0));
        if (x < 0.0 && k > lo) hi = k - 1;
        else if (x >= de && k < hi) lo = k + 1;
        else break;   // the root lies on this segment (or on the continued end segment)
        t = it < 8 ? (ek + x - eos.e_min) * inv_de : (double)((lo + hi) >> 1);
    }
    const double pe = fma(c, x, pk);
    const double w = 1.0 / (E + pe);
    p = (T)pe;
    cs2 = (T)c;
    v2 = (T)(m2 * w * w);
    winv = (T)(w * sc);
}

// a3 for a state with its own sound speed (tabulated closure):
//   a_d = ( |v_d| (1-cs2) + sqrt(cs2 (1-v^2)(1 - v_d^2 - (v^2 - v_d^2) cs2)) ) / (1 - v^2 cs2)
template <class T>
HD T signal_speed_cs(T vd, T v2, T cs2) {
    const T vd2 = vd * vd;
    const T disc = max_nonneg(cs2 * ((T)1 - v2) * ((T)1 - vd2 - (v2 - vd2) * cs2), (T)0);
    return (tabs(vd) * ((T)1 - cs2) + tsqrt(disc)) / ((T)1 - v2 * cs2);
}

// a3. directional characteristic speeds, c_s^2 = 1/3 (a3):
//   a_d = ( |v_d| (1-cs2) + cs sqrt((1-v^2)(1 - v_d^2 - (v^2 - v_d^2) cs2)) ) / (1 - v^2 cs2)
// FLOOR = false: for states known to be well inside |v| < 1 (the branch-free MUSTA path), where disc > 0 holds with
// a wide margin and the floor is dead weight.
template <class T, bool FLOOR = true>
HD T signal_speed(T vd, T v2, T inv_den) {
    const T cs2 = (T)(1.0 / 3.0);
    const T cs = (T)0.57735026918962576451;
    const T vd2 = vd * vd;
    // disc >= 0 analytically; the floor keeps the reciprocal-square-root seed finite when a clamped state
    // (reading Q16) drives it to zero
    T disc = ((T)1 - v2) * ((T)1 - vd2 - (v2 - vd2) * cs2);
    if (FLOOR) disc = max_nonneg(disc, (T)1e-30);   // (a negative value loses too)
    return (tabs(vd) * ((T)1 - cs2) + cs * fast_sqrt(disc)) * inv_den;
}
template <class T>
HD T speed_inv_den(T v2) { return fast_rcp(tfma(v2, (T)(-1.0 / 3.0), (T)1)); }

// ------------------------------------------------------------------------------------------------
// a7. WENO reconstructions in numerator/denominator form.
// For stencil values f_0..f_{2r-2} (upwind-ordered) the reconstructed value at the interface is
//   f_c + N / D,   f_c = the centre value f_{r-1},
// with N = sum_k d_k P_k (q_k - f_c) and D = sum_k d_k P_k, P_k = prod_{j != k} (eps' + beta'_j)^2:
// the classic weights alpha_k = d_k/(eps+beta_k)^2 multiplied through by prod_j (eps+beta_j)^2
// (DESIGN.md section 6).  beta' and eps' carry a common scale factor, which cancels in N/D.

// Cross-multiplied weights need the products prod_{j != k} B_j^2 (B^4 for WENO5, B^6 for WENO7) to stay inside the
// normal range.  fp64: they do for |data| < 1e25 (documented in include/hydro.h).  fp32: flux jumps of order 1e3
// overflow B^6 and a tiny epsilon on flat data underflows it, so the B_k are first multiplied by the power of two
// that brings the smallest of them to [1, 2) (exact, and it cancels in N/D) and clamped at 2^17 (WENO7; 2^25 for
// WENO5): a sub-stencil whose indicator is 2^17 times the smallest carries a weight below 2^-34 of the dominant one
// either way, far under fp32 resolution; the products then stay below 2^102, which leaves room for the factors g_k.
template <class T, int NB>
HD void normalise_indicators(T (&B)[NB]) {}
#ifdef __CUDA_ARCH__
template <>
__device__ __forceinline__ void normalise_indicators<float, 3>(float (&B)[3]) {
    const float m = fminf(B[0], fminf(B[1], B[2]));
    // 2^(127 - exponent(m)); the exponent field is held at 253 so that s stays a normal positive number when the
    // smallest indicator is 2^127 or beyond (or Inf): s = 0 would zero every B_k and N / D would be 0 / 0
    const float s = __int_as_float(0x7f000000 - min(__float_as_int(m) & 0x7f800000, 0x7e800000));
    // WENO5 takes B only to the 4th power: the clamp can sit at 2^25 (products below 2^100)
    const float cap = 33554432.0f;   // 2^25
#pragma unroll
    for (int k = 0; k < 3; ++k) B[k] = fminf(B[k] * s, cap);
}
template <>
__device__ __forceinline__ void normalise_indicators<float, 4>(float (&B)[4]) {
    const float m = fminf(fminf(B[0], B[1]), fminf(B[2], B[3]));
    const float s = __int_as_float(0x7f000000 - min(__float_as_int(m) & 0x7f800000, 0x7e800000));
    const float cap = 131072.0f;     // 2^17
#pragma unroll
    for (int k = 0; k < 4; ++k) B[k] = fminf(B[k] * s, cap);
}
#endif

// WENO5 (Jiang-Shu, O3) from the four first differences D_j = f_{j+1} - f_j of the stencil
// (a, b, c, d, e).  Here beta' = 4 beta and eps4 = 4 eps.
template <class T>
HD void weno5_nd_d(T D1, T D2, T D3, T D4, T eps4, T& N, T& D) {
    const T t0 = D2 - D1, t1 = D3 - D2, t2 = D4 - D3;      // second differences
    const T u0 = tfma((T)3, D2, -D1);                      // a - 4b + 3c
    const T u1 = D2 + D3;                                  // d - b
    const T u2 = tfma((T)-3, D3, D4);                      // 3c - 4d + e, sign irrelevant (squared)
    // (13/3) t^2 as the square of sqrt(13/3) t: a fused multiply-add with a repeated operand reads two registers
    // instead of three and issues in 2 cycles instead of 3
    const T rk = (T)2.0816659994661327353;   // sqrt(13/3)
    const T s0_ = rk * t0, s1_ = rk * t1, s2_ = rk * t2;
    T B[3];
    B[0] = tfma(s0_, s0_, tfma(u0, u0, eps4));
    B[1] = tfma(s1_, s1_, tfma(u1, u1, eps4));
    B[2] = tfma(s2_, s2_, tfma(u2, u2, eps4));
    normalise_indicators<T, 3>(B);
    const T s0 = B[0] * B[0], s1 = B[1] * B[1], s2 = B[2] * B[2];
    const T P0 = s1 * s2, P1 = s0 * s2, P2 = s0 * s1;
    // 10 d_k = (1, 6, 3);  q_k - c = (5 D2 - 2 D1)/6, (D2 + 2 D3)/6, (4 D3 - D4)/6
    const T g0 = tfma((T)(5.0 / 6.0), D2, (T)(-1.0 / 3.0) * D1);
    const T g1 = tfma((T)2, D3, D2);                       // times 6 d1/(6) = 1
    const T g2 = tfma((T)2, D3, (T)-0.5 * D4);             // (4 D3 - D4)/6 * 3
    N = tfma(P0, g0, tfma(P1, g1, P2 * g2));
    D = tfma((T)6, P1, tfma((T)3, P2, P0));
}
template <class T>
HD void weno5_nd(T a, T b, T c, T d, T e, T eps4, T& N, T& D) {
    weno5_nd_d(b - a, c - b, d - c, e - d, eps4, N, D);
}

// WENO7 (Balsara-Shu, O4).  For the cubic through four cell averages written as
// c0 + c1 x + c2 x^2 + c3 x^3 about the centre of cell i (dx = 1) the smoothness indicator is
//   beta = (c1 + c3/4)^2 + (13/3) c2^2 + (781/20) c3^2
// (the integrals of the squared first, second and third derivatives over the cell, summed); in terms
// of undivided differences c3 = D3/6, c2 = (second difference at i)/2 and c1 follows from matching
// the averages.  This equals the integer-coefficient quadratic forms of O4 divided by 240.
// Input: the six first differences E_j = f_{j+1} - f_j of the stencil (a..g), centre cell d.
template <class T>
HD void weno7_nd_d(T E1, T E2, T E3, T E4, T E5, T E6, T eps, T& N, T& D) {
    const T S1 = E2 - E1, S2 = E3 - E2, S3 = E4 - E3, S4 = E5 - E4, S5 = E6 - E5;  // second
    const T T1 = S2 - S1, T2 = S3 - S2, T3 = S4 - S3, T4 = S5 - S4;                // third
    // Stencil k holds cells (k..k+3) of (a..g); the centre cell d sits at position 3-k inside it.
    // Solving "cell averages of the cubic = stencil values" for the coefficients about cell d gives
    // (checked with exact rationals against the 240-beta forms of O4, and q_k against O4's q_k):
    //   k=0: c3 = T1/6, c2 = (S2 + T1)/2, c1 + c3/4 = E3 + S2/2 + T1/3
    //   k=1: c3 = T2/6, c2 = S3/2,        c1 + c3/4 = (E3 + E4)/2 - T2/6
    //   k=2: c3 = T3/6, c2 = S3/2,        c1 + c3/4 = (E3 + E4)/2 - T3/6
    //   k=3: c3 = T4/6, c2 = (S4 - T4)/2, c1 + c3/4 = E4 - S4/2 + T4/3
    // the factors 13/3 and 781/20 go into the coefficients as their square roots, so that every term of an
    // indicator is the square of ONE value: a fused multiply-add with a repeated operand reads two registers
    // instead of three and issues in 2 cycles instead of 3
    const T r13 = (T)2.0816659994661327353, r781 = (T)6.2489999199871975245;   // sqrt(13/3), sqrt(781/20)
    const T c3s = r781 * (T)(1.0 / 6.0), c2s = r13 * (T)0.5;
    const T c3_0 = T1 * c3s, c2_0 = c2s * (S2 + T1), m_0 = E3 + tfma((T)0.5, S2, (T)(1.0 / 3.0) * T1);
    const T c3_1 = T2 * c3s, c2_1 = c2s * S3, m_1 = tfma((T)(-1.0 / 6.0), T2, (T)0.5 * (E3 + E4));
    const T c3_2 = T3 * c3s, c2_2 = c2_1, m_2 = tfma((T)(-1.0 / 6.0), T3, (T)0.5 * (E3 + E4));
    const T c3_3 = T4 * c3s, c2_3 = c2s * (S4 - T4), m_3 = E4 + tfma((T)-0.5, S4, (T)(1.0 / 3.0) * T4);
    T B[4];
    B[0] = tfma(m_0, m_0, tfma(c2_0, c2_0, tfma(c3_0, c3_0, eps)));
    B[1] = tfma(m_1, m_1, tfma(c2_1, c2_1, tfma(c3_1, c3_1, eps)));
    B[2] = tfma(m_2, m_2, tfma(c2_2, c2_2, tfma(c3_2, c3_2, eps)));
    B[3] = tfma(m_3, m_3, tfma(c2_3, c2_3, tfma(c3_3, c3_3, eps)));
    normalise_indicators<T, 4>(B);
    const T s0 = B[0] * B[0], s1 = B[1] * B[1], s2 = B[2] * B[2], s3 = B[3] * B[3];
    const T s01 = s0 * s1, s23 = s2 * s3;
    const T P0 = s1 * s23, P1 = s0 * s23, P2 = s01 * s3, P3 = s01 * s2;
    // q_k - d (centre value) from the candidate polynomials of O4:
    //   q0 - d = (-3a + 13b - 23c + 13d)/12 = (13 E3 - 10 E2 + 3 E1)/12
    //   q1 - d = (b - 5c + d + 3e)/12       = (3 E4 + 4 E3 - E2)/12
    //   q2 - d = (-c - 5d + 7e - f)/12      = (-E5 + 6 E4 + E3)/12
    //   q3 - d = (-9d + 13e - 5f + g)/12    = (E6 - 4 E5 + 9 E4)/12
    // 35 d_k = (1, 12, 18, 4)
    const T g0 = tfma((T)(13.0 / 12.0), E3, tfma((T)(-10.0 / 12.0), E2, (T)(3.0 / 12.0) * E1));
    const T g1 = tfma((T)3, E4, tfma((T)4, E3, -E2));                        // x 12/12
    const T g2 = tfma((T)9, E4, tfma((T)1.5, E3, (T)-1.5 * E5));             // x 18/12
    const T g3 = tfma((T)3, E4, tfma((T)(-4.0 / 3.0), E5, (T)(1.0 / 3.0) * E6)); // x 4/12
    N = tfma(P0, g0, tfma(P1, g1, tfma(P2, g2, P3 * g3)));
    D = tfma((T)12, P1, tfma((T)18, P2, tfma((T)4, P3, P0)));
}
template <class T>
HD void weno7_nd(T a, T b, T c, T d, T e, T f, T g, T eps, T& N, T& D) {
    weno7_nd_d(b - a, c - b, d - c, e - d, f - e, g - f, eps, N, D);
}

}  // namespace hydro
