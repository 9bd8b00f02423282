// kernel_musta.cuh -- stage kernels of MUSTA-FORCE (a7'): L(u) of Eq. (2) fused with
// the SSP-RK3 combination (a9), every interface flux computed once.
//
// The predictor-corrector flux runs con2prim on face states that mix all five fields, so one thread carries all
// five fields of its stencil.
//   musta_xz_kernel<T>     x and z fluxes in ONE marching kernel without block barriers.  A warp is a row of 32
//       consecutive x positions (lane 0 is the helper column one cell below the 31 cells the warp owns), a block is
//       four such rows, and every thread marches along z through a chunk of planes:
//         z: the 4-cell stencil of the thread's column lives in a register window;
//         x: the plane-k cells of the window are exactly the row the x-stencil needs, so every lane writes its cell
//            into a per-WARP shared-memory row, 3 halo lanes add the cells beyond the row's ends, and after a
//            __syncwarp each lane reads its 4-cell x-stencil from that row.  The lower-face flux comes from lane-1
//            by shuffle.
//       Writes Uout = ca u^n + cb (u_s + dt (L_x + L_z)).
//   musta_y_kernel<T, EPI> the marching sweep along y: thread per (x, z) column, threads of a warp along x (so every
//       access is coalesced), adds cb dt L_y to Uout.  EPI (stage 3 of a CFL step): the thread holds the finished
//       cell, so it also reduces the max signal speed of the new state (a4) for the next step's dt.
// Every global read of the marching loops is a cp.async into the thread's own slots, DEPTH cells ahead (pipeline.cuh).
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

// 4-cell stencil of the five conserved fields of one column, in registers (all indices compile-time constants)
template <class T>
struct MustaWindow {
    T uu[NF][MUSTA_M];
    __device__ __forceinline__ T u(int c, int k) const { return uu[c][k]; }
    __device__ __forceinline__ void put(int m, const T v[NF]) {
#pragma unroll
        for (int c = 0; c < NF; ++c) uu[c][m] = v[c];
    }
    __device__ __forceinline__ void shift() {
#pragma unroll
        for (int m = 0; m + 1 < MUSTA_M; ++m) {
#pragma unroll
            for (int c = 0; c < NF; ++c) uu[c][m] = uu[c][m + 1];
        }
    }
};

// stencil accessor into a shared-memory row: conserved field c of stencil cell k at ub[c * astride + k]
template <class T>
struct RowAcc {
    const T* ub;
    int astride;
    __device__ __forceinline__ T u(int c, int k) const { return ub[c * astride + k]; }
};

// FAST: the default configuration (K = 2, minmod, p = e/3) with everything a compile-time constant; otherwise the
// run-time K / limiter / closure.  The choice is made per KERNEL, not per interface: with both bodies inlined the
// marching loops outgrew the instruction cache (stall reason "no instruction").
template <class T, int DIR, bool FAST, class Acc>
__device__ __forceinline__ void musta_iface(const Acc& acc, const StageArgs& A, T fh[NF], int& flag) {
    if (FAST) musta_force_stages<T, DIR, 2, 0>(acc, 2, (T)A.musta_C, 0, 0, (T)0, fh, flag);
    else musta_force_stages<T, DIR, 0, -1>(acc, A.musta_K, (T)A.musta_C, A.limiter, A.eos.kind, (T)A.eos.p0, fh, flag);
}
inline bool musta_fast(const StageArgs& A) { return A.musta_K == 2 && A.limiter == 0 && A.eos.kind == 0; }

// ---------------------------------------------------------------------------------------------------------
template <class T>
struct MustaXZShape {
    static constexpr int R = MUSTA_R, D = MUSTA_DEPTH;
    static constexpr int NS = NF + NF;                       // window cell k+R, u^n of plane k: slots per thread
    static constexpr int NHL = 2 * R - 1;                    // halo lanes: R-1 cells below, R cells above the row
    static constexpr int RWX = 32 + 2 * R - 1;               // cells of a row with halo
    static constexpr int STAGE = NS * MUSTA_THREADS + MUSTA_ROWS * NHL * NF;
    // pipeline stages, the warps' rows, and one parking slot per thread and field for the last z-flux
    static constexpr size_t smem_bytes() {
        return sizeof(T) * ((size_t)D * STAGE + MUSTA_ROWS * NF * RWX + NF * MUSTA_THREADS);
    }
};

template <class T, bool FAST>
__global__ void __launch_bounds__(MUSTA_THREADS, 3)
musta_xz_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* Un, T* Uout, Ctl* ctl, int zc) {
    using S = MustaXZShape<T>;
    constexpr int R = S::R, M = 2 * R, NS = S::NS, NHL = S::NHL, RWX = S::RWX, D = S::D, TH = MUSTA_THREADS;
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
    const int k0 = (int)blockIdx.z * zc;
    const int k1 = min(k0 + zc, G.n[2]);
    const long long p0 = G.pidx(il, j, k0);
    const long long ph = G.pidx(min(hcell, imax), j, k0);
    const bool use_un = A.mode != 1 && A.ca != 0.0;
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

    MustaWindow<T> zw;
    T nxt[NF];
#pragma unroll
    for (int m = 0; m < M; ++m) {   // cells k0-R .. k0+R-1
#pragma unroll
        for (int c = 0; c < NF; ++c) nxt[c] = __ldg(Us + c * G.fs + p0 + (long long)(m - R) * G.sxy);
        zw.put(m, nxt);
    }
    // the helper lane and the idle lanes of a ragged last tile march through x-ghost columns, whose z-ghost cells
    // are edge ghosts nobody fills: their z-fluxes are discarded, and so must be their unphysical-state flag
    int zflag = 0;
    {
        T f0[NF];
        musta_iface<T, 2, FAST>(zw, A, f0, zflag);   // face k0 - 1/2
#pragma unroll
        for (int c = 0; c < NF; ++c) park[c * TH] = f0[c];
    }
    const T dt = (T)ctl->dt, ca = (T)A.ca, cb = (T)A.cb, inv_dx = (T)A.inv_dx;

    for (int k = k0; k < k1; ++k) {
        cp_async_wait<D - 1>();   // plane k's stage has landed
        const T* st = sm + ((k - k0) % D) * S::STAGE;
        const T* src = st + tid;
        T hv[NF];
#pragma unroll
        for (int c = 0; c < NF; ++c) nxt[c] = src[c * TH];
        if (lane < NHL) {
            const T* hs = st + NS * TH + (wy * NHL + lane) * NF;
#pragma unroll
            for (int c = 0; c < NF; ++c) hv[c] = hs[c];
        }
        zw.shift();
        zw.put(M - 1, nxt);
        __syncwarp();             // every lane is done with the row of plane k-1
#pragma unroll
        for (int c = 0; c < NF; ++c) row[c * RWX + lane + R - 1] = zw.uu[c][R - 1];
        if (lane < NHL) {
#pragma unroll
            for (int c = 0; c < NF; ++c) row[c * RWX + hq] = hv[c];
        }
        __syncwarp();
        T L[NF], f[NF];
        musta_iface<T, 2, FAST>(zw, A, f, zflag);
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            L[c] = park[c * TH] - f[c];
            park[c * TH] = f[c];
        }
#pragma unroll
        for (int c = 0; c < NF; ++c) f[c] = (T)0;
        if (need_x) {
            RowAcc<T> acc{row + lane, RWX};
            musta_iface<T, 0, FAST>(acc, A, f, flag);
        }
#pragma unroll
        for (int c = 0; c < NF; ++c) L[c] += shfl_up1<T>(f[c]) - f[c];
        if (own) {
            const long long q = p0 + (long long)(k - k0) * G.sxy;
            if (A.mode == 1) {
#pragma unroll
                for (int c = 0; c < NF; ++c) Uout[c * G.fs + q] = L[c] * inv_dx;
            } else {
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    T v = tfma(dt, L[c] * inv_dx, zw.uu[c][R - 1]);
                    if (use_un) v = tfma(ca, src[(NF + c) * TH], cb * v);   // u^n: read late, it is only needed here
                    Uout[c * G.fs + q] = v;
                }
            }
        }
        issue(k + D);             // refill the slot just consumed
    }
    if (flag || (own && zflag)) ctl->flag = 1;
}

// ---------------------------------------------------------------------------------------------------------
template <class T>
constexpr size_t musta_y_smem_bytes() {
    return sizeof(T) * ((size_t)MUSTA_DEPTH * (NF + NF) + NF) * MUSTA_THREADS;
}

template <class T, bool EPI, bool FAST>
__global__ void __launch_bounds__(MUSTA_THREADS, 4)
musta_y_kernel(Geom G, StageArgs A, const T* __restrict__ Us, T* Uout, Ctl* ctl, int yc) {
    constexpr int R = MUSTA_R, M = 2 * R, NVO = NF + NF, D = MUSTA_DEPTH, TH = MUSTA_THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);   // [D][NVO][TH], then [NF][TH]
    const int tid = threadIdx.x + 32 * threadIdx.y;
    T* park = sm + D * NVO * TH + tid;
    const int i = blockIdx.x * 32 + threadIdx.x;
    const int kz = blockIdx.y * MUSTA_ROWS + threadIdx.y;
    // lanes beyond the grid leave; the ballot (taken while the warp is whole) is the mask of the final reduction
    const unsigned wmask = __ballot_sync(0xffffffffu, i < G.n[0] && kz < G.n[2]);
    if (i >= G.n[0] || kz >= G.n[2]) return;
    const long long ms = G.sx;
    const int j0 = (int)blockIdx.z * yc;
    const int j1 = min(j0 + yc, G.n[1]);
    const long long p0 = G.pidx(i, j0, kz);
    int flag = 0;
    auto issue = [&](int j) {
        if (j < j1) {
            T* dst = sm + ((j - j0) % D) * NVO * TH + tid;
            const long long q = p0 + (long long)(j - j0) * ms;
            const long long qr = q + (long long)R * ms;
#pragma unroll
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + c * TH, Us + c * G.fs + qr);
#pragma unroll
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + (NF + c) * TH, Uout + c * G.fs + q);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d < D; ++d) issue(j0 + d);

    MustaWindow<T> zw;
    T nxt[NF];
#pragma unroll
    for (int m = 0; m < M; ++m) {
#pragma unroll
        for (int c = 0; c < NF; ++c) nxt[c] = __ldg(Us + c * G.fs + p0 + (long long)(m - R) * ms);
        zw.put(m, nxt);
    }
    {
        T f0[NF];
        musta_iface<T, 1, FAST>(zw, A, f0, flag);
#pragma unroll
        for (int c = 0; c < NF; ++c) park[c * TH] = f0[c];
    }
    const T coef = A.mode == 1 ? (T)A.inv_dx : (T)(A.cb * ctl->dt * A.inv_dx);
    double amax = 0.0;
    for (int j = j0; j < j1; ++j) {
        T f[NF], o[NF];
        cp_async_wait<D - 1>();   // the oldest stage (cell j) has landed
        const T* src = sm + ((j - j0) % D) * NVO * TH + tid;
#pragma unroll
        for (int c = 0; c < NF; ++c) nxt[c] = src[c * TH];
        zw.shift();
        zw.put(M - 1, nxt);
        musta_iface<T, 1, FAST>(zw, A, f, flag);
        const long long q = p0 + (long long)(j - j0) * ms;
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            o[c] = tfma(coef, park[c * TH] - f[c], src[(NF + c) * TH]);   // old output: read late
            Uout[c * G.fs + q] = o[c];
            park[c * TH] = f[c];
        }
        issue(j + D);             // refill the slot just consumed
        if (EPI) {   // a4 of the finished cell (all three axes are active whenever this kernel runs)
            T w[NW];
            prim_of_cell(o, w, flag, A.eos);
            amax = fmax(amax, fmax((double)w[W_AX], fmax((double)w[W_AX + 1], (double)w[W_AX + 2])));
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

// stage = x/z kernel (writes Uout) + y sweep (adds L_y; stage 3 of a CFL step: the max signal speed of the new state)
template <class T>
int launch_musta(const Geom& G, const StageArgs& A, const T* Us, const T* Un, T* Uout, Ctl* ctl, int zc, int yc,
                 cudaStream_t st, int* launches, char* err, size_t errlen) {
    const dim3 b(32, MUSTA_ROWS, 1);
    const dim3 g((G.n[0] + 30) / 31, (G.n[1] + MUSTA_ROWS - 1) / MUSTA_ROWS, (G.n[2] + zc - 1) / zc);
    const dim3 gy((G.n[0] + 31) / 32, (G.n[2] + MUSTA_ROWS - 1) / MUSTA_ROWS, (G.n[1] + yc - 1) / yc);
    const size_t sxz = MustaXZShape<T>::smem_bytes(), sy = musta_y_smem_bytes<T>();
    const bool epi = A.epi_max && A.mode != 1;
    if (musta_fast(A)) {
        musta_xz_kernel<T, true><<<g, b, sxz, st>>>(G, A, Us, Un, Uout, ctl, zc);
        if (epi) musta_y_kernel<T, true, true><<<gy, b, sy, st>>>(G, A, Us, Uout, ctl, yc);
        else musta_y_kernel<T, false, true><<<gy, b, sy, st>>>(G, A, Us, Uout, ctl, yc);
    } else {
        musta_xz_kernel<T, false><<<g, b, sxz, st>>>(G, A, Us, Un, Uout, ctl, zc);
        if (epi) musta_y_kernel<T, true, false><<<gy, b, sy, st>>>(G, A, Us, Uout, ctl, yc);
        else musta_y_kernel<T, false, false><<<gy, b, sy, st>>>(G, A, Us, Uout, ctl, yc);
    }
    *launches = 2;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(err, errlen, "%s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

}  // namespace hydro
