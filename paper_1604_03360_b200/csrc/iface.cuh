// iface.cuh -- one interface flux (steps a5..a7 and a7') from a stencil accessor.
//
// The accessor hides where the stencil lives (global memory in the generic kernel, the shared-memory
// ring / plane in the fused kernel): acc.u(c, k) is conserved field c of stencil cell k and
// acc.w(a, k) primitive array a (W_V + axis, W_P, W_AX + axis), k = 0 .. 2r-1 for cells i-r+1 .. i+r.
#pragma once
#include "device_math.cuh"

namespace hydro {

template <class T> struct is_f64 { static constexpr bool value = false; };
template <> struct is_f64<double> { static constexpr bool value = true; };

// value of (f+ reconstruction) + (f- reconstruction) from the two N/D pairs and the centre values.
// fp64: one reciprocal for the pair.  fp32: the product of the two denominators can leave the
// normal range, so two hardware reciprocals.
template <class T>
HD T combine_pair(T centre, T Np, T Dp, T Nm, T Dm) {
    if (is_f64<T>::value) {
        const T num = tfma(Np, Dm, Nm * Dp);
        return tfma(num, fast_rcp(Dp * Dm), centre);
    } else {
        return tfma(Np, fast_rcp(Dp), tfma(Nm, fast_rcp(Dm), centre));
    }
}

// alpha as the plain maximum of a_DIR over the 2r stencil cells of an accessor with w(W_AX + DIR, k)
template <class T, int M, int DIR, class Acc>
HD T alpha_of_cells(const Acc& acc) {
    T al = acc.w(W_AX + DIR, 0);
#pragma unroll
    for (int k = 1; k < M; ++k) al = max_nonneg(al, acc.w(W_AX + DIR, k));
    return al;
}

// a5-a7. Component-wise local Lax-Friedrichs flux with WENO_r reconstruction at interface i+1/2 along
// axis DIR (O5, reading Q3):
//   alpha = max_k a_d(k);  f+-_k = (F_d(u_k) +- alpha u_k)/2;
//   fhat = WENO(f+ on cells 0..2r-2) + WENO(f- on cells 2r-1..1, mirrored).
// The factor 1/2 is pulled out of the reconstruction: WENO is homogeneous of degree one when eps is
// scaled with the square of the data, WENO_eps(g/2) = WENO_{4 eps}(g)/2, exactly in binary floating
// point.  With v_d = M_d * winv the split fluxes are u (v_d +- alpha) for the fields that are simply
// advected (M_j, j != d, and R), M_d (v_d +- alpha) + p for j = d, and M_d +- alpha E for E.
// Returns TWICE the interface flux: the caller folds the 1/2 into its 1/dx factor (exact in binary floating point).
// alpha comes from the accessor (acc.alpha<DIR, 2r>()): a stencil in registers carries pair maxima, the others take the
// maximum of the 2r values.
template <class T, int R, int DIR, class Acc>
HD void llf_weno_iface2(const Acc& acc, T eps, T fh[NF]) {
    constexpr int M = 2 * R;
    constexpr int I5 = (R == 4) ? 5 : 3, I6 = (R == 4) ? 6 : 4;  // only read when R == 4
    T md[M], vp[M], vm[M];
    const T al = acc.template alpha<DIR, M>();
#pragma unroll
    for (int k = 0; k < M; ++k) {
        md[k] = acc.u(1 + DIR, k);
        const T vd = acc.w(W_V + DIR, k);
        vp[k] = vd + al;
        vm[k] = vd - al;
    }
    // eps scale: weno5_nd works with 4*beta(g) = 16*beta(g/2); weno7_nd with beta(g) = 4*beta(g/2)
    const T epsx = (R == 3 ? (T)16 : (T)4) * eps;
#pragma unroll
    for (int c = 0; c < NF; ++c) {
        T fp[M - 1], fm[M - 1];
        if (c == 0) {
#pragma unroll
            for (int k = 0; k < M - 1; ++k) {
                fp[k] = tfma(al, acc.u(0, k), md[k]);
                fm[k] = tfma(-al, acc.u(0, M - 1 - k), md[M - 1 - k]);
            }
        } else if (c == 1 + DIR) {
#pragma unroll
            for (int k = 0; k < M - 1; ++k) {
                fp[k] = tfma(md[k], vp[k], acc.w(W_P, k));
                fm[k] = tfma(md[M - 1 - k], vm[M - 1 - k], acc.w(W_P, M - 1 - k));
            }
        } else {
#pragma unroll
            for (int k = 0; k < M - 1; ++k) {
                fp[k] = acc.u(c, k) * vp[k];
                fm[k] = acc.u(c, M - 1 - k) * vm[M - 1 - k];
            }
        }
        T Np, Dp, Nm, Dm;
        if (R == 3) {
            weno5_nd(fp[0], fp[1], fp[2], fp[3], fp[4], epsx, Np, Dp);
            weno5_nd(fm[0], fm[1], fm[2], fm[3], fm[4], epsx, Nm, Dm);
        } else {
            weno7_nd(fp[0], fp[1], fp[2], fp[3], fp[4], fp[I5], fp[I6], epsx, Np, Dp);
            weno7_nd(fm[0], fm[1], fm[2], fm[3], fm[4], fm[I5], fm[I6], epsx, Nm, Dm);
        }
        fh[c] = combine_pair(fp[R - 1] + fm[R - 1], Np, Dp, Nm, Dm);
    }
}
// ------------------------------------------------------------------------------------------------
// a7'. MUSTA-FORCE flux with MUSCL/minmod data (O6, O7; readings Q6-Q8).
template <class T>
HD T minmod(T a, T b) {
    if (a * b <= (T)0) return (T)0;
    const T m = tmin(tabs(a), tabs(b));
    return a > (T)0 ? m : -m;
}
#ifdef __CUDA_ARCH__
// fp64 on the device: the same function on the bit patterns, in the integer pipe (an fp64 compare, select or |x|
// occupies the fp64 pipe, which is the one this path is bound by).  Doubles are sign-magnitude, so among two doubles
// of the SAME sign the one of smaller magnitude is the smaller one as a signed 64-bit integer, whatever that sign:
// minmod = opposite signs ? 0 : min_s64(a, b).  Differs from the product test only when a*b underflows (both |a|,
// |b| < 1e-154), where it returns that tiny slope instead of 0, and for a zero operand, where it returns +-0.
template <>
__device__ __forceinline__ double minmod<double>(double a, double b) {
    const long long ia = __double_as_longlong(a), ib = __double_as_longlong(b);
    const long long m = ia < ib ? ia : ib;
    return __longlong_as_double((ia ^ ib) < 0 ? 0ll : m);
}
#endif

// The other limiters ("a variety of slope limiting methods", a7'): limited slope
// of the backward difference a and the forward difference b.  1 van Leer 2ab/(a+b); 2 MC
// sign(a) min(2|a|, 2|b|, |a+b|/2); 3 superbee sign(a) max(min(2|a|,|b|), min(|a|,2|b|)); all 0 unless ab > 0.
template <class T>
HD T limited_slope(int lim, T a, T b) {
    if (lim == 0) return minmod(a, b);
    if (a * b <= (T)0) return (T)0;
    const T aa = tabs(a), ab = tabs(b);
    if (lim == 1) return (T)2 * a * b * fast_rcp(aa + ab) * (a > (T)0 ? (T)1 : (T)-1);
    T m;
    if (lim == 2) m = tmin(tmin((T)2 * aa, (T)2 * ab), (T)0.5 * (aa + ab));
    else m = tmax(tmin((T)2 * aa, ab), tmin(aa, (T)2 * ab));
    return a > (T)0 ? m : -m;
}

// physical flux of a conserved state along DIR plus its signal speed (every evaluation needs its own
// con2prim, O7).  Q is modified only if the Q16 clamp fires.  EOSRT: the equation of state is the run-time
// (eos, p0); otherwise the default p = e/3 at compile time.
template <class T, int DIR, bool EOSRT>
HD void flux_and_speed(const T Q[NF], T F[NF], T& a, int& flag, const EosArgs& eos) {
    T winv, p, v2, cs2 = (T)0;
    if (EOSRT && eos.kind == 1) con2prim_p0(Q[0], Q[1], Q[2], Q[3], (T)eos.p0, winv, p, v2, flag);
    else if (EOSRT && eos.kind == 2) con2prim_tab(Q[0], Q[1], Q[2], Q[3], eos, winv, p, v2, cs2, flag);
    else con2prim(Q[0], Q[1], Q[2], Q[3], winv, p, v2, flag);
    const T vd = Q[1 + DIR] * winv;
    F[0] = Q[1 + DIR];
#pragma unroll
    for (int j = 0; j < 3; ++j) F[1 + j] = (j == DIR) ? tfma(Q[1 + j], vd, p) : Q[1 + j] * vd;
    F[4] = Q[4] * vd;
    if (EOSRT && eos.kind == 1) a = tabs(vd);
    else if (EOSRT && eos.kind == 2) a = signal_speed_cs(vd, v2, cs2);
    else a = signal_speed(vd, v2, speed_inv_den(v2));
}
template <class T, int DIR, bool EOSRT>
HD void flux_only(const T Q[NF], T F[NF], int& flag, const EosArgs& eos) {
    T winv, p, v2, cs2;
    if (EOSRT && eos.kind == 1) con2prim_p0(Q[0], Q[1], Q[2], Q[3], (T)eos.p0, winv, p, v2, flag);
    else if (EOSRT && eos.kind == 2) con2prim_tab(Q[0], Q[1], Q[2], Q[3], eos, winv, p, v2, cs2, flag);
    else con2prim(Q[0], Q[1], Q[2], Q[3], winv, p, v2, flag);
    const T vd = Q[1 + DIR] * winv;
    F[0] = Q[1 + DIR];
#pragma unroll
    for (int j = 0; j < 3; ++j) F[1 + j] = (j == DIR) ? tfma(Q[1 + j], vd, p) : Q[1 + j] * vd;
    F[4] = Q[4] * vd;
}

// The same two evaluations for the default closure p = e/3, arranged for the predictor-corrector loop, which runs six
// of them per interface: ONE test sends every state the Q16 clamp could touch (E below the floor, |M| > (1 - 1e-12) E,
// NaN) to the general functions above, so the common path carries no clamp selects; it needs one reciprocal,
// 1/(2E+s) -- the pressure is (s - E)/3, whose cancellation error, an ulp of E, is an ulp of the flux it enters.
template <class T, int DIR, bool SPEED>
HD void musta_flux(const T Q[NF], T F[NF], T& a, int& flag) {
    const T E = Q[0];
    const T m2 = tfma(Q[1], Q[1], tfma(Q[2], Q[2], Q[3] * Q[3]));
    const T t = E * E;
    const T c2 = ((T)1 - (T)1e-12) * ((T)1 - (T)1e-12);
    if (below_floor(E) || !(m2 <= c2 * t)) {   // rare (kept inline: out of line, Q and F would live in local memory)
        const EosArgs gas = {0, 0.0, nullptr, 0, 0.0, 1.0};
        if (SPEED) flux_and_speed<T, DIR, false>(Q, F, a, flag, gas);
        else flux_only<T, DIR, false>(Q, F, flag, gas);
        return;
    }
    const T s = fast_sqrt(tfma((T)4, t, (T)-3 * m2));
    const T w = (T)3 * fast_rcp(tfma((T)2, E, s));   // v_i = M_i w
    const T p = (s - E) * (T)(1.0 / 3.0);
    const T vd = Q[1 + DIR] * w;
    F[0] = Q[1 + DIR];
#pragma unroll
    for (int j = 0; j < 3; ++j) F[1 + j] = (j == DIR) ? tfma(Q[1 + j], vd, p) : Q[1 + j] * vd;
    F[4] = Q[4] * vd;
    if (SPEED) {
        const T v2 = m2 * w * w;
        a = signal_speed(vd, v2, speed_inv_den(v2));
    }
}

// Limited slope of a cell from its backward and forward differences (O6); LIMS == 0: minmod at compile time.
template <class T, int LIMS>
HD T musta_slope(int lim, T dm, T dp) { return LIMS == 0 ? minmod(dm, dp) : limited_slope(lim, dm, dp); }

// The predictor-corrector loop (O7, readings Q7, Q8) from the two face states, general form: every con2prim carries
// the Q16 clamp, K and the closure may be run-time values.  QL, QR are overwritten by the corrected states.
// KS > 0: the number of stages is the compile-time constant KS; KS = 0: run-time K.
template <class T, int DIR, int KS, bool EOSRT>
HD void musta_force_core(T QL[NF], T QR[NF], int K, T C, const EosArgs& eos, T fh[NF], int& flag) {
    const T invC = fast_rcp(C);   // (one MUFU-seeded reciprocal per interface; a true division costs a subroutine)
    const int nst = KS > 0 ? KS : K;
#pragma unroll
    for (int stage = 1; stage <= nst; ++stage) {
        T FL[NF], FR[NF], QM[NF], FM[NF], aL, aR;
        if (EOSRT) {
            flux_and_speed<T, DIR, true>(QL, FL, aL, flag, eos);
            flux_and_speed<T, DIR, true>(QR, FR, aR, flag, eos);
        } else {
            musta_flux<T, DIR, true>(QL, FL, aL, flag);
            musta_flux<T, DIR, true>(QR, FR, aR, flag);
        }
        const T S = max_nonneg(aL, aR);
        // p = p0: S = max |v_d| vanishes where the fluid is at rest and tau = C/S is then infinite, in the oracle
        // as here (reading Q7 has no finite local step without a sound speed): MUSTA-FORCE with that closure is
        // for moving fluid only
        const T tau = C * fast_rcp(S), itau = S * invC;
#pragma unroll
        for (int c = 0; c < NF; ++c) QM[c] = (T)0.5 * ((QL[c] + QR[c]) - tau * (FR[c] - FL[c]));
        if (EOSRT) flux_only<T, DIR, true>(QM, FM, flag, eos);
        else {
            T unused;
            musta_flux<T, DIR, false>(QM, FM, unused, flag);
        }
#pragma unroll
        for (int c = 0; c < NF; ++c)
            fh[c] = (T)0.25 * (FL[c] + (T)2 * FM[c] + FR[c] - (QR[c] - QL[c]) * itau);
        if (stage < nst) {
#pragma unroll
            for (int c = 0; c < NF; ++c) {
                QL[c] = QL[c] - tau * (fh[c] - FL[c]);
                QR[c] = QR[c] - tau * (FR[c] - fh[c]);
            }
        }
    }
}

// acc.u(c, k), k = 0..3 for cells i-1 .. i+2.  K stages, local Courant number C (tau = C/S).
// LIMS >= 0: the limiter is the compile-time constant LIMS and the closure the default one; LIMS < 0: run-time
// limiter and closure.
template <class T, int DIR, int KS, int LIMS, class Acc>
HD void musta_force_stages(const Acc& acc, int K, T C, int lim, const EosArgs& eos, T fh[NF], int& flag) {
    constexpr bool EOSRT = LIMS < 0;
    T QL[NF], QR[NF];
#pragma unroll
    for (int c = 0; c < NF; ++c) {
        const T u0 = acc.u(c, 0), u1 = acc.u(c, 1), u2 = acc.u(c, 2), u3 = acc.u(c, 3);
        const T dm = u1 - u0, d0 = u2 - u1, dp = u3 - u2;
        QL[c] = tfma((T)0.5, musta_slope<T, LIMS>(lim, dm, d0), u1);
        QR[c] = tfma((T)-0.5, musta_slope<T, LIMS>(lim, d0, dp), u2);
    }
    musta_force_core<T, DIR, KS, EOSRT>(QL, QR, K, C, eos, fh, flag);
}

// ------------------------------------------------------------------------------------------------
// The same loop for the default configuration (p = e/3, compile-time K), arranged for the fp64 pipe (DESIGN.md
// section 6); the marching kernels use it.  It is ONE basic block: no clamp, no branch, so that the compiler can
// interleave the independent evaluations F(Q_L), F(Q_R) of a stage and the two interfaces a thread works on.  A state
// the Q16 clamp could touch (E below the floor or not finite, |M| close to or above E, NaN) only sets `bad`; the
// caller then discards the result and runs the general form above on the same face states.
//
// Rearrangements (rounding only): with G_L = Q_L + tau F_L and G_R = Q_R - tau F_R,
//   2 Q_M = G_L + G_R,   F(2 Q_M) = 2 F(Q_M)  (the flux is homogeneous of degree one in Q, exactly so in binary
//   floating point),   4 F* = (F_L + Q_L/tau) + (F_R - Q_R/tau) + F(2 Q_M) = (G_L - G_R)/tau + F(2 Q_M),
//   corrector: Q_L' = G_L - (tau/4)(4 F*),  Q_R' = G_R + (tau/4)(4 F*).
// Returns FOUR TIMES the flux: the caller folds the 1/4 into its 1/dx factor (exact).
// Admissibility of the states the branch-free path evaluates, accumulated over an interface as ONE running minimum
// (a register, not a chain of booleans): after all evaluations `margin >= 0` must hold.
//   fp64 (integer pipe, high words): margin = min over the states of  hi(E) - hi(1e-300) - 1  and
//   hi(D) - hi(t) - 2, with D = 4 E^2 - 3 M^2 and t = E^2: hi(D) >= hi(t) + 2 means D > t (1 + 2^-21), i.e.
//   |M| < (1 - 1e-7) E, well inside the Q16 bound; a negative E or D is a negative integer.  Infinities and NaNs can
//   pass here: they make the flux non-finite, which musta_force_fast4 tests once at its end.
//   fp32: the same two margins as floating-point differences.
template <class T> struct MustaMargin { T m; };
template <> struct MustaMargin<double> { int m; };
template <class T>
HD void musta_margin_init(MustaMargin<T>& g) { g.m = (T)1; }
template <class T>
HD void musta_margin(MustaMargin<T>& g, T E, T t, T D) {
    g.m = tmin(g.m, tmin(E - (T)1e-30, D - t * (T)1.0001));
    if (!(D <= (T)3e38)) g.m = (T)-1;
}
template <class T>
HD bool musta_margin_bad(const MustaMargin<T>& g) { return !(g.m >= (T)0); }
template <class T>
HD bool musta_finite(T x) { return tabs(x) <= (T)3e38; }
#ifdef __CUDA_ARCH__
template <>
__device__ __forceinline__ void musta_margin_init<double>(MustaMargin<double>& g) { g.m = 0x7fffffff; }
template <>
__device__ __forceinline__ void musta_margin<double>(MustaMargin<double>& g, double E, double t, double D) {
    g.m = min(g.m, min(__double2hiint(E) - 0x01a56e20, __double2hiint(D) - __double2hiint(t) - 2));
}
template <>
__device__ __forceinline__ bool musta_margin_bad<double>(const MustaMargin<double>& g) { return g.m < 0; }
template <>
__device__ __forceinline__ bool musta_finite<double>(double x) {
    return (unsigned)(__double2hiint(x) << 1) < 0xffe00000u;
}
#endif

template <class T, int DIR, bool SPEED>
HD void musta_eval_fast(const T Q[NF], T F[NF], T& a, MustaMargin<T>& g) {
    const T E = Q[0], md = Q[1 + DIR];
    const T m2 = tfma(Q[1], Q[1], tfma(Q[2], Q[2], Q[3] * Q[3]));
    const T t = E * E;
    const T D = tfma((T)4, t, (T)-3 * m2);
    musta_margin(g, E, t, D);
    const T s = fast_sqrt(D);
    const T w = (T)3 * fast_rcp(tfma((T)2, E, s));   // v_i = M_i w
    const T p = (s - E) * (T)(1.0 / 3.0);            // cancellation error: an ulp of E, i.e. an ulp of the flux it enters
    const T vd = md * w;
    F[0] = md;
#pragma unroll
    for (int j = 0; j < 3; ++j) F[1 + j] = (j == DIR) ? tfma(Q[1 + j], vd, p) : Q[1 + j] * vd;
    F[4] = Q[4] * vd;
    if (SPEED) {
        const T v2 = m2 * w * w;
        a = signal_speed<T, false>(vd, v2, speed_inv_den(v2));
    }
}

template <class T, int DIR, int KS>
HD void musta_force_fast4(const T QL0[NF], const T QR0[NF], T C, T invC, T fh4[NF], bool& bad) {
    T QL[NF], QR[NF];
    MustaMargin<T> g;
    musta_margin_init(g);
#pragma unroll
    for (int c = 0; c < NF; ++c) {
        QL[c] = QL0[c];
        QR[c] = QR0[c];
    }
#pragma unroll
    for (int stage = 1; stage <= KS; ++stage) {
        T FL[NF], FR[NF], GL[NF], GR[NF], Q2[NF], F2[NF], aL, aR, unused;
        musta_eval_fast<T, DIR, true>(QL, FL, aL, g);
        musta_eval_fast<T, DIR, true>(QR, FR, aR, g);
        const T S = max_nonneg(aL, aR);
        const T tau = C * fast_rcp(S), itau = S * invC;
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            GL[c] = tfma(tau, FL[c], QL[c]);
            GR[c] = tfma(-tau, FR[c], QR[c]);
            Q2[c] = GL[c] + GR[c];
        }
        musta_eval_fast<T, DIR, false>(Q2, F2, unused, g);
        // (F_L + Q_L/tau) + (F_R - Q_R/tau) = (G_L - G_R)/tau
#pragma unroll
        for (int c = 0; c < NF; ++c) fh4[c] = tfma(itau, GL[c] - GR[c], F2[c]);
        if (stage < KS) {
            const T t4 = (T)0.25 * tau;
#pragma unroll
            for (int c = 0; c < NF; ++c) {
                QL[c] = tfma(-t4, fh4[c], GL[c]);
                QR[c] = tfma(t4, fh4[c], GR[c]);
            }
        }
    }
    // a NaN or an infinity anywhere above has reached the flux
    bad = musta_margin_bad(g) || !musta_finite(((fh4[0] + fh4[1]) + (fh4[2] + fh4[3])) + fh4[4]);
}

template <class T, int DIR, class Acc>
HD void musta_force_iface(const Acc& acc, int K, T C, int lim, const EosArgs& eos, T fh[NF], int& flag) {
    if (K == 2 && lim == 0 && eos.kind == 0) musta_force_stages<T, DIR, 2, 0>(acc, K, C, lim, eos, fh, flag);
    else musta_force_stages<T, DIR, 0, -1>(acc, K, C, lim, eos, fh, flag);
}

}  // namespace hydro
