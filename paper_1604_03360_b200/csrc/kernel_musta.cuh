// kernel_musta.cuh -- stage kernels of MUSTA-FORCE (a7'): L(u) of Eq. (2) fused with
// the SSP-RK3 combination (a9), every interface flux computed once.
//
// The predictor-corrector flux runs con2prim on face states that mix all five fields, so one thread carries all
// five fields of its stencil.  The MUSCL slope belongs to a cell and is made once per cell.
//   musta_xz_kernel<T, FAST>  x and z fluxes in ONE marching kernel without block barriers.  A warp is a row of 32
//       consecutive x positions (lane 0 is the helper column one cell below the 31 cells the warp owns), a block is
//       four such rows, and every thread marches along z through a chunk of planes:
//         z: the column state (MustaColumn: u_k, u_{k+1}, their difference, Q_L of face k+1/2) lives in registers;
//         x: every lane writes its plane-k cell into a per-WARP shared-memory row, 3 halo lanes add the cells beyond
//            the row's ends; after a __syncwarp each lane reads its two neighbours, makes the slope of ITS cell,
//            keeps Q_L of its upper face and hands Q_R of its lower face to the lane below by shuffle (the last
//            lane also makes the one slope beyond the row).  The lower-face flux comes from lane-1 by shuffle.
//         The x and the z interface of a plane are evaluated in one basic block (four independent con2prim chains).
//       Writes Uout = ca u^n + cb (u_s + dt (L_x + L_z)).
//   musta_y_kernel<T, EPI, FAST>  the marching sweep along y: thread per (x, z) column, threads of a warp along x (so
//       every access is coalesced), two cells per iteration, adds cb dt L_y to Uout.  EPI (stage 3 of a CFL step):
//       the thread holds the finished cells, so it also reduces the max signal speed of the new state (a4).
// FAST = the default configuration (K = 2, minmod, p = e/3): the branch-free core of iface.cuh with the general,
// clamped core as the rare repair; otherwise the general core with run-time K, limiter and closure.
// Every global read of the marching loops is a cp.async into the thread's own slots, a few cells ahead (pipeline.cuh).
#pragma once
#include <cstdio>

#include "grid.cuh"
#include "iface.cuh"
#include "kernel_generic.cuh"
#include "kernels_aux.cuh"
#include "pipeline.cuh"

namespace hydro {

constexpr int MUSTA_DEPTH = 3;   // cells in flight per thread
constexpr int MUSTA_ROWS = 4;    // warps per block
constexpr int MUSTA_THREADS = 32 * MUSTA_ROWS;
constexpr int MUSTA_R = 2, MUSTA_M = 4;

// Marching state of one column along the marched axis: the MUSCL slope (O6) belongs to a CELL, so it is made once per
// cell and serves both of the cell's faces.  With cell m the one whose upper face is being computed:
//   u0 = u_m, u1 = u_{m+1}, db = u_{m+1} - u_m, ql = Q_L of face m+1/2 = u_m + slope_m / 2.
// advance(u2) takes u_{m+2}, makes slope_{m+1} and returns Q_R of face m+1/2 = u_{m+1} - slope_{m+1}/2; commit() then
// moves on to cell m+1.
template <class T, int LIMS>
struct MustaColumn {
    T u0[NF], u1[NF], db[NF], ql[NF];
    T df[NF], qn[NF];   // between advance() and commit(): u_{m+2} - u_{m+1}, Q_L of face m+3/2
    __device__ __forceinline__ void init(const T a[NF], const T b[NF], const T c[NF], int lim) {   // cells m-1, m, m+1
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            u0[f] = b[f];
            u1[f] = c[f];
            db[f] = c[f] - b[f];
            ql[f] = tfma((T)0.5, musta_slope<T, LIMS>(lim, b[f] - a[f], db[f]), b[f]);
        }
    }
    __device__ __forceinline__ void advance(const T u2[NF], int lim, T qr[NF]) {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            df[f] = u2[f] - u1[f];
            const T h = (T)0.5 * musta_slope<T, LIMS>(lim, db[f], df[f]);
            qr[f] = u1[f] - h;
            qn[f] = u1[f] + h;
        }
    }
    __device__ __forceinline__ void commit(const T u2[NF]) {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            u0[f] = u1[f];
            u1[f] = u2[f];
            db[f] = df[f];
            ql[f] = qn[f];
        }
    }
};

// FAST: the default configuration (K = 2, minmod, p = e/3) with everything a compile-time constant and the branch-free
// core (iface.cuh); otherwise the run-time K / limiter / closure.  The choice is made per KERNEL, not per interface:
// with both bodies inlined the marching loops outgrew the instruction cache (stall reason "no instruction").
inline bool musta_fast(const StageArgs& A) { return A.musta_K == 2 && A.limiter == 0 && A.eos.kind == 0; }

// general form on a copy of the face states; returns four times the flux like the fast core
template <class T, int DIR, bool FAST>
__device__ __forceinline__ void musta_general4(const T QL[NF], const T QR[NF], const StageArgs& A, T C, T f4[NF],
                                               int& flag) {
    T a[NF], b[NF];
#pragma unroll
    for (int c = 0; c < NF; ++c) {
        a[c] = QL[c];
        b[c] = QR[c];
    }
    if (FAST) musta_force_core<T, DIR, 2, false>(a, b, 2, C, A.eos, f4, flag);
    else musta_force_core<T, DIR, 0, true>(a, b, A.musta_K, C, A.eos, f4, flag);
#pragma unroll
    for (int c = 0; c < NF; ++c) f4[c] *= (T)4;
}

// ---------------------------------------------------------------------------------------------------------
template <class T>
struct MustaXZShape {
    static constexpr int R = MUSTA_R, D = MUSTA_DEPTH;
    static constexpr int NS = NF + NF;                       // cell k+R, u^n of plane k: slots per thread
    static constexpr int NHL = 2 * R - 1;                    // halo lanes: R-1 cells below, R cells above the row
    static constexpr int RWX = 32 + 2 * R - 1;               // cells of a row with halo
    static constexpr int STAGE = NS * MUSTA_THREADS + MUSTA_ROWS * NHL * NF;
    // pipeline stages, the warps' rows, and one parking slot per thread and field for the last z-flux
    static constexpr size_t smem_bytes() {
        return sizeof(T) * ((size_t)D * STAGE + MUSTA_ROWS * NF * RWX + NF * MUSTA_THREADS);
    }
};

#ifndef MUSTA_XZ_MINB
#define MUSTA_XZ_MINB 2
#endif
#ifndef MUSTA_Y_MINB
#define MUSTA_Y_MINB 2
#endif

template <class T, bool FAST>
__global__ void __launch_bounds__(MUSTA_THREADS, MUSTA_XZ_MINB)
musta_xz_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* Un, T* Uout, Ctl* ctl, int zc) {
    using S = MustaXZShape<T>;
    constexpr int R = S::R, NS = S::NS, NHL = S::NHL, RWX = S::RWX, D = S::D, TH = MUSTA_THREADS;
    constexpr int LIMS = FAST ? 0 : -1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);
    const int lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32 + lane;
    const int i0 = (int)blockIdx.x * 31 - 1, i = i0 + lane;
    const int j = (int)blockIdx.y * MUSTA_ROWS + wy;
    if (j >= G.n[1]) return;   // whole warp
    T* row = sm + D * S::STAGE + wy * NF * RWX;              // [NF][RWX], this warp's
    T* park = sm + D * S::STAGE + MUSTA_ROWS * NF * RWX + tid;   // [NF][TH]: this thread's last z-flux
    const bool own = lane >= 1 && i < G.n[0];
    const bool need_x = i < G.n[0];                        // i >= -1 always
    const int imax = G.n[0] - 1 + G.g[0];
    const int il = min(i, imax);                           // column this lane loads (idle lanes: clamped)
    const int hcell = lane < R - 1 ? i0 - (R - 1) + lane : i0 + 32 + (lane - (R - 1));   // halo lanes' column
    const int hq = lane < R - 1 ? lane : 32 + lane;        // and its position in the row
    const int k0 = A.kbeg + (int)blockIdx.z * zc;
    const int k1 = min(k0 + zc, A.kend);
    const long long p0 = G.pidx(il, j, k0);
    const long long ph = G.pidx(min(hcell, imax), j, k0);
    const bool use_un = A.mode != 1 && A.ca != 0.0;
    const int lim = A.limiter;
    const T C = (T)A.musta_C, invC = fast_rcp(C);
    int flag = 0;

    auto issue = [&](int k) {
        if (k < k1) {
            T* st = sm + ((k - k0) % D) * S::STAGE;
            T* dst = st + tid;
            const long long q = p0 + (long long)(k - k0) * G.sxy, qr = q + (long long)R * G.sxy;
#pragma unroll
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + c * TH, Us + c * G.fs + qr);
            if (use_un) {
#pragma unroll
                for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + (NF + c) * TH, Un + c * G.fs + q);
            }
            if (lane < NHL) {
                T* hd = st + NS * TH + (wy * NHL + lane) * NF;
                const long long qh = ph + (long long)(k - k0) * G.sxy;
#pragma unroll
                for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(hd + c, Us + c * G.fs + qh);
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d < D; ++d) issue(k0 + d);

    // the helper lane and the idle lanes of a ragged last tile march through x-ghost columns, whose z-ghost cells
    // are edge ghosts nobody fills: their z-fluxes are discarded, and so must be their unphysical-state flag
    int zflag = 0;
    MustaColumn<T, LIMS> zc_;
    {   // face k0 - 1/2 from cells k0-2 .. k0+1, then the column state of cell k0
        T c[4][NF];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
#pragma unroll
            for (int f = 0; f < NF; ++f) c[m][f] = __ldg(Us + f * G.fs + p0 + (long long)(m - R) * G.sxy);
        }
        zc_.init(c[0], c[1], c[2], lim);   // column at cell k0-1: ql = Q_L of face k0-1/2
        T qr[NF], f0[NF];
        zc_.advance(c[3], lim, qr);
        if (FAST) {
            bool bad = false;
            musta_force_fast4<T, 2, 2>(zc_.ql, qr, C, invC, f0, bad);
            if (bad) musta_general4<T, 2, FAST>(zc_.ql, qr, A, C, f0, zflag);
        } else {
            musta_general4<T, 2, FAST>(zc_.ql, qr, A, C, f0, zflag);
        }
        zc_.commit(c[3]);
#pragma unroll
        for (int f = 0; f < NF; ++f) park[f * TH] = f0[f];
    }
    // the interface functions return four times the flux: the 1/4 of the FORCE average goes into dt/dx
    const T dtdx = (T)(A.mode == 1 ? 0.25 * A.inv_dx : 0.25 * ctl->dt * A.inv_dx), ca = (T)A.ca, cb = (T)A.cb;

    for (int k = k0; k < k1; ++k) {
        cp_async_wait<D - 1>();   // plane k's stage has landed
        const T* st = sm + ((k - k0) % D) * S::STAGE;
        const T* src = st + tid;
        T u2[NF];
#pragma unroll
        for (int c = 0; c < NF; ++c) u2[c] = src[c * TH];
        __syncwarp();             // every lane is done with the row of plane k-1
#pragma unroll
        for (int c = 0; c < NF; ++c) row[c * RWX + lane + R - 1] = zc_.u0[c];
        if (lane < NHL) {         // the halo cells go from their slots straight into the row
            const T* hs = st + NS * TH + (wy * NHL + lane) * NF;
#pragma unroll
            for (int c = 0; c < NF; ++c) row[c * RWX + hq] = hs[c];
        }
        __syncwarp();
        // z: face k + 1/2
        T qrz[NF], qlx[NF], qrx[NF];
        zc_.advance(u2, lim, qrz);
        // x: this lane's cell makes its slope once, keeps Q_L of its upper face and hands Q_R of its lower face to
        // the lane below; the last lane makes the slope of the first cell beyond the row as well
        {
            T up[NF], dp[NF];
#pragma unroll
            for (int c = 0; c < NF; ++c) {
                const T um = row[c * RWX + lane + R - 2];
                up[c] = row[c * RWX + lane + R];
                dp[c] = up[c] - zc_.u0[c];
                const T h = (T)0.5 * musta_slope<T, LIMS>(lim, zc_.u0[c] - um, dp[c]);
                qlx[c] = zc_.u0[c] + h;
                qrx[c] = __shfl_down_sync(0xffffffffu, zc_.u0[c] - h, 1);
            }
            if (lane == 31) {
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    const T upp = row[c * RWX + lane + R + 1];
                    qrx[c] = tfma((T)-0.5, musta_slope<T, LIMS>(lim, dp[c], upp - up[c]), up[c]);
                }
            }
        }
        T fz[NF], fx[NF];
        if (FAST) {   // both interfaces in one basic block; the rare repairs afterwards
            bool badz = false, badx = false;
            musta_force_fast4<T, 2, 2>(zc_.ql, qrz, C, invC, fz, badz);
            musta_force_fast4<T, 0, 2>(qlx, qrx, C, invC, fx, badx);
            if (badz) musta_general4<T, 2, FAST>(zc_.ql, qrz, A, C, fz, zflag);
            if (badx && need_x) musta_general4<T, 0, FAST>(qlx, qrx, A, C, fx, flag);
        } else {
            musta_general4<T, 2, FAST>(zc_.ql, qrz, A, C, fz, zflag);
            int xf = 0;
            musta_general4<T, 0, FAST>(qlx, qrx, A, C, fx, xf);
            if (need_x) flag |= xf;
        }
        T L[NF];
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            L[c] = (park[c * TH] - fz[c]) + (shfl_up1<T>(fx[c]) - fx[c]);
            park[c * TH] = fz[c];
        }
        if (own) {
            const long long q = p0 + (long long)(k - k0) * G.sxy;
            if (A.mode == 1) {
#pragma unroll
                for (int c = 0; c < NF; ++c) Uout[c * G.fs + q] = L[c] * dtdx;
            } else {
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    T v = tfma(dtdx, L[c], zc_.u0[c]);
                    if (use_un) v = tfma(ca, src[(NF + c) * TH], cb * v);   // u^n: read late, it is only needed here
                    Uout[c * G.fs + q] = v;
                }
            }
        }
        zc_.commit(u2);
        issue(k + D);             // refill the slot just consumed
    }
    if (flag || (own && zflag)) ctl->flag = 1;
}

// ---------------------------------------------------------------------------------------------------------
// The y sweep advances TWO cells per iteration: the two interfaces j+1/2 and j+3/2 are independent, and in one basic
// block they give the fp64 pipe four independent con2prim chains (two face states each) to interleave; a dependent fp64
// instruction issues only every 8 cycles, and more warps do not replace that instruction-level parallelism
// (DESIGN.md section 8).
constexpr int MUSTA_YG = 2;      // cp.async groups in flight, two cells each
template <class T>
constexpr size_t musta_y_smem_bytes() {
    return sizeof(T) * ((size_t)2 * MUSTA_YG * (NF + NF) + NF) * MUSTA_THREADS;
}

template <class T, bool EPI, bool FAST>
__global__ void __launch_bounds__(MUSTA_THREADS, MUSTA_Y_MINB)
musta_y_kernel(Geom G, StageArgs A, const T* __restrict__ Us, T* Uout, Ctl* ctl, int yc) {
    constexpr int R = MUSTA_R, NVO = NF + NF, TH = MUSTA_THREADS, NG = MUSTA_YG;
    constexpr int LIMS = FAST ? 0 : -1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);   // [NG][2][NVO][TH], then [NF][TH]
    const int tid = threadIdx.x + 32 * threadIdx.y;
    T* park = sm + 2 * NG * NVO * TH + tid;
    const int i = blockIdx.x * 32 + threadIdx.x;
    const int kz = blockIdx.y * MUSTA_ROWS + threadIdx.y;
    // lanes beyond the grid leave; the ballot (taken while the warp is whole) is the mask of the final reduction
    const unsigned wmask = __ballot_sync(0xffffffffu, i < G.n[0] && kz < G.n[2]);
    if (i >= G.n[0] || kz >= G.n[2]) return;
    const long long ms = G.sx;
    const int j0 = (int)blockIdx.z * yc;
    const int j1 = min(j0 + yc, G.n[1]);
    const long long p0 = G.pidx(i, j0, kz);
    const int lim = A.limiter;
    const T C = (T)A.musta_C, invC = fast_rcp(C);
    int flag = 0;
    // group g = cells j0 + 2g, j0 + 2g + 1: per cell the stencil cell R ahead and the old output
    auto issue = [&](int g) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int j = j0 + 2 * g + h;
            if (j < j1) {
                T* dst = sm + ((g % NG) * 2 + h) * NVO * TH + tid;
                const long long q = p0 + (long long)(j - j0) * ms;
                const long long qr = q + (long long)R * ms;
#pragma unroll
                for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + c * TH, Us + c * G.fs + qr);
#pragma unroll
                for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + (NF + c) * TH, Uout + c * G.fs + q);
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int g = 0; g < NG; ++g) issue(g);

    MustaColumn<T, LIMS> col;
    {   // face j0 - 1/2 from cells j0-2 .. j0+1, then the column state of cell j0
        T c[4][NF];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
#pragma unroll
            for (int f = 0; f < NF; ++f) c[m][f] = __ldg(Us + f * G.fs + p0 + (long long)(m - R) * ms);
        }
        col.init(c[0], c[1], c[2], lim);
        T qr[NF], f0[NF];
        col.advance(c[3], lim, qr);
        if (FAST) {
            bool bad = false;
            musta_force_fast4<T, 1, 2>(col.ql, qr, C, invC, f0, bad);
            if (bad) musta_general4<T, 1, FAST>(col.ql, qr, A, C, f0, flag);
        } else {
            musta_general4<T, 1, FAST>(col.ql, qr, A, C, f0, flag);
        }
        col.commit(c[3]);
#pragma unroll
        for (int f = 0; f < NF; ++f) park[f * TH] = f0[f];
    }
    // four times the flux comes in
    const T coef = A.mode == 1 ? (T)(0.25 * A.inv_dx) : (T)(0.25 * A.cb * ctl->dt * A.inv_dx);
    double amax = 0.0;
    const int ng = (j1 - j0 + 1) / 2;
    for (int g = 0; g < ng; ++g) {
        const int j = j0 + 2 * g;
        const bool second = j + 1 < j1;   // an odd chunk ends on a half group: its second cell is computed on stale
                                          // slots and thrown away
        cp_async_wait<NG - 1>();          // the oldest group has landed
        const T* src = sm + (g % NG) * 2 * NVO * TH + tid;
        T ua[NF], ub[NF], qla[NF], qra[NF], qlb[NF], qrb[NF], fa[NF], fb[NF];
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            ua[c] = src[c * TH];
            ub[c] = src[(NVO + c) * TH];
            qla[c] = col.ql[c];
        }
        col.advance(ua, lim, qra);
        col.commit(ua);
#pragma unroll
        for (int c = 0; c < NF; ++c) qlb[c] = col.ql[c];
        col.advance(ub, lim, qrb);
        col.commit(ub);
        if (FAST) {   // both interfaces in one basic block; the rare repairs afterwards
            bool bada = false, badb = false;
            musta_force_fast4<T, 1, 2>(qla, qra, C, invC, fa, bada);
            musta_force_fast4<T, 1, 2>(qlb, qrb, C, invC, fb, badb);
            if (bada) musta_general4<T, 1, FAST>(qla, qra, A, C, fa, flag);
            if (badb && second) musta_general4<T, 1, FAST>(qlb, qrb, A, C, fb, flag);
        } else {
            musta_general4<T, 1, FAST>(qla, qra, A, C, fa, flag);
            int f2 = 0;
            musta_general4<T, 1, FAST>(qlb, qrb, A, C, fb, f2);
            if (second) flag |= f2;
        }
        const long long q = p0 + (long long)(j - j0) * ms;
        T oa[NF], ob[NF];
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            oa[c] = tfma(coef, park[c * TH] - fa[c], src[(NF + c) * TH]);   // old output: read late
            Uout[c * G.fs + q] = oa[c];
        }
        if (second) {
#pragma unroll
            for (int c = 0; c < NF; ++c) {
                ob[c] = tfma(coef, fa[c] - fb[c], src[(NVO + NF + c) * TH]);
                Uout[c * G.fs + q + ms] = ob[c];
                park[c * TH] = fb[c];
            }
        }
        issue(g + NG);            // refill the slots just consumed
        if (EPI) {   // a4 of the finished cells (all three axes are active whenever this kernel runs)
            amax = fmax(amax, (double)max_speed_of_cell(oa, A.eos, true, true, true, flag));
            if (second) amax = fmax(amax, (double)max_speed_of_cell(ob, A.eos, true, true, true, flag));
        }
    }
    if (EPI) warp_max_to(amax, &ctl->maxspeed_next_bits, wmask);
    if (flag) ctl->flag = 1;
}

template <class T>
int configure_musta(char* err, size_t errlen) {
    const int sxz = (int)MustaXZShape<T>::smem_bytes(), sy = (int)musta_y_smem_bytes<T>();
    const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
    cudaError_t e = cudaFuncSetAttribute(musta_xz_kernel<T, true>, attr, sxz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(musta_xz_kernel<T, false>, attr, sxz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(musta_y_kernel<T, false, true>, attr, sy);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(musta_y_kernel<T, true, true>, attr, sy);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(musta_y_kernel<T, false, false>, attr, sy);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(musta_y_kernel<T, true, false>, attr, sy);
    if (e != cudaSuccess) {
        snprintf(err, errlen, "cudaFuncSetAttribute (musta): %s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

// stage = x/z kernel over the planes [A.kbeg, A.kend) (writes Uout) + y sweep (adds L_y; stage 3 of a CFL step: the
// max signal speed of the new state).  parts: bit 0 the x/z kernel, bit 1 the y sweep.
template <class T>
int launch_musta(const Geom& G, const StageArgs& A, const T* Us, const T* Un, T* Uout, Ctl* ctl, int zc, int yc,
                 cudaStream_t st, int parts, int* launches, char* err, size_t errlen) {
    const dim3 b(32, MUSTA_ROWS, 1);
    const size_t sxz = MustaXZShape<T>::smem_bytes(), sy = musta_y_smem_bytes<T>();
    const bool epi = A.epi_max && A.mode != 1;
    *launches = 0;
    if ((parts & 1) && A.kend > A.kbeg) {
        const dim3 g((G.n[0] + 30) / 31, (G.n[1] + MUSTA_ROWS - 1) / MUSTA_ROWS, (A.kend - A.kbeg + zc - 1) / zc);
        if (musta_fast(A)) musta_xz_kernel<T, true><<<g, b, sxz, st>>>(G, A, Us, Un, Uout, ctl, zc);
        else musta_xz_kernel<T, false><<<g, b, sxz, st>>>(G, A, Us, Un, Uout, ctl, zc);
        ++*launches;
    }
    if (parts & 2) {
        const dim3 gy((G.n[0] + 31) / 32, (G.n[2] + MUSTA_ROWS - 1) / MUSTA_ROWS, (G.n[1] + yc - 1) / yc);
        if (musta_fast(A)) {
            if (epi) musta_y_kernel<T, true, true><<<gy, b, sy, st>>>(G, A, Us, Uout, ctl, yc);
            else musta_y_kernel<T, false, true><<<gy, b, sy, st>>>(G, A, Us, Uout, ctl, yc);
        } else {
            if (epi) musta_y_kernel<T, true, false><<<gy, b, sy, st>>>(G, A, Us, Uout, ctl, yc);
            else musta_y_kernel<T, false, false><<<gy, b, sy, st>>>(G, A, Us, Uout, ctl, yc);
        }
        ++*launches;
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(err, errlen, "%s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

}  // namespace hydro
