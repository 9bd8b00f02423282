// kernel_weno.cuh -- stage kernels of the WENO schemes: L(u) of Eq. (2) fused with
// the SSP-RK3 combination (a9) and with con2prim + signal speeds + the CFL max of the finished cells
// (a2-a4); every interface flux computed once.
//
//   weno_xz_kernel<T, R>        x and z fluxes in ONE marching kernel without block barriers.  A warp is a row of 32
//       consecutive x positions (lane 0 is the helper column one cell below the 31 cells the warp owns), a block is
//       four such rows, and every thread marches along z through a chunk of planes:
//         z: the 2r-cell stencil of the thread's column lives in a register window (conserved fields, v_z, p, a_z);
//         x: the plane-k cells of the window are exactly the row the x-stencil needs, so every lane writes its own
//            (conserved, v_x, p, a_x) into a per-WARP shared-memory row, 2r-1 halo lanes add the cells beyond the
//            row's ends, and after a __syncwarp each lane reads its 2r-cell x-stencil from that row.  The lower-face
//            flux comes from lane-1 by shuffle.
//       Writes Uout = ca u^n + cb (u_s + dt (L_x + L_z)).
//   weno_y_kernel<T, R, EPI>    the marching sweep along y: thread per (x, z) column, threads of a warp along x (so
//       every access is coalesced), adds cb dt L_y to Uout.  EPI (Runge-Kutta mode): the thread holds the finished
//       stage value of its cell, so it also makes the next stage's primitives W' = (v, p, a_x, a_y, a_z) of that
//       cell (a2-a3; written to the OTHER W buffer, this stage's W is still being read by neighbouring blocks) and,
//       in stage 3, the max signal speed of the new state (a4): no separate con2prim pass over the grid.
// Every global read of the marching loops is a cp.async into the thread's own slots DEPTH cells ahead (pipeline.cuh).
//
// Performance model of these kernels (measured with the microbenchmarks quoted there): an fp64
// warp-instruction holds its scheduler's issue port for 2 cycles, a DFMA with three distinct register operands for 3,
// and EVERY other instruction adds one more cycle: the kernels are bound by their total instruction count, not by
// occupancy, so what matters here is to issue as few instructions as possible per interface.
#pragma once
#include <cstdio>

#include "grid.cuh"
#include "iface.cuh"
#include "kernel_generic.cuh"
#include "kernels_aux.cuh"
#include "pipeline.cuh"

namespace hydro {

#ifndef WENO5_MINB
#define WENO5_MINB 3
#endif
constexpr int WENO_ZC = 64, WENO_YC = 128;   // default cells per chunk of the z / y march ("tile_zc" / "sweep_zc")
constexpr int WENO_DEPTH = 3;                // cells in flight per thread
constexpr int WENO_ROWS = 4;                 // warps per block
constexpr int WENO_THREADS = 32 * WENO_ROWS;

// stencil of one column along the marched axis DIR, in registers: cells m-R+1 .. m+R, per cell the five conserved
// fields and v_DIR, p; of a_DIR the maxima of neighbouring pairs (alpha is then the maximum of R of them: one new
// maximum per cell instead of 2R-1 per interface).  All indices are compile-time constants after unrolling.
template <class T, int R, int DIR>
struct WenoWindow {
    static constexpr int M = 2 * R, NV = NF + 3;
    T uu[NF][M], ww[2][M], pm[M - 1], a_last;
    __device__ __forceinline__ T u(int c, int k) const { return uu[c][k]; }
    __device__ __forceinline__ T w(int a, int k) const { return ww[a == W_P ? 1 : 0][k]; }
    template <int D2, int M2>
    __device__ __forceinline__ T alpha() const {
        T al = pm[0];
#pragma unroll
        for (int k = 2; k < M - 1; k += 2) al = max_nonneg(al, pm[k]);
        return al;
    }
    static __device__ __forceinline__ void fetch(T v[NV], const T* __restrict__ U, const T* __restrict__ W,
                                                 long long fs, long long q) {
#pragma unroll
        for (int c = 0; c < NF; ++c) v[c] = __ldg(U + c * fs + q);
        v[NF + 0] = __ldg(W + (W_V + DIR) * fs + q);
        v[NF + 1] = __ldg(W + W_P * fs + q);
        v[NF + 2] = __ldg(W + (W_AX + DIR) * fs + q);
    }
    __device__ __forceinline__ void first(const T v[NV]) {   // cell 0 of an empty window
#pragma unroll
        for (int c = 0; c < NF; ++c) uu[c][0] = v[c];
        ww[0][0] = v[NF];
        ww[1][0] = v[NF + 1];
        a_last = v[NF + 2];
    }
    __device__ __forceinline__ void put(int m, const T v[NV]) {   // cell m >= 1, after cell m-1
#pragma unroll
        for (int c = 0; c < NF; ++c) uu[c][m] = v[c];
        ww[0][m] = v[NF];
        ww[1][m] = v[NF + 1];
        pm[m - 1] = max_nonneg(a_last, v[NF + 2]);
        a_last = v[NF + 2];
    }
    __device__ __forceinline__ void shift() {
#pragma unroll
        for (int m = 0; m + 1 < M; ++m) {
#pragma unroll
            for (int c = 0; c < NF; ++c) uu[c][m] = uu[c][m + 1];
            ww[0][m] = ww[0][m + 1];
            ww[1][m] = ww[1][m + 1];
        }
#pragma unroll
        for (int m = 0; m + 2 < M; ++m) pm[m] = pm[m + 1];
    }
};

// x-stencil accessor into the warp's shared-memory row: arrays u[5], v_x, p, a_x with pitch `pitch`
template <class T>
struct XRowAcc {
    const T* b;
    int pitch;
    __device__ __forceinline__ T u(int c, int k) const { return b[c * pitch + k]; }
    __device__ __forceinline__ T w(int a, int k) const { return b[(NF + (a == W_P ? 1 : (a >= W_AX ? 2 : 0))) * pitch + k]; }
    template <int DIR, int M>
    __device__ __forceinline__ T alpha() const { return alpha_of_cells<T, M, DIR>(*this); }
};

// ---------------------------------------------------------------------------------------------------------
template <class T, int R>
struct WenoXZShape {
    using Win = WenoWindow<T, R, 2>;
    static constexpr int NV = Win::NV;                        // window cell: conserved, v_z, p, a_z
    static constexpr int NS = NV + 2 + NF;                    // + v_x, a_x and u^n of plane k
    static constexpr int NH = NF + 3;                         // row arrays: conserved, v_x, p, a_x
    static constexpr int NHL = 2 * R - 1;                     // halo lanes: R-1 cells below, R cells above the row
    static constexpr int RWX = 32 + 2 * R - 1;                // cells of a row with halo
    static constexpr int STAGE = NS * WENO_THREADS + WENO_ROWS * NHL * NH;
    // pipeline stages, the warps' rows, and one parking slot per thread and field for the last z-flux (it is
    // only needed once per plane; parked, the kernel fits its register budget without spilling)
    static constexpr size_t smem_bytes() {
        return sizeof(T) * ((size_t)WENO_DEPTH * STAGE + WENO_ROWS * NH * RWX + NF * WENO_THREADS);
    }
};

template <class T, int R>
__global__ void __launch_bounds__(WENO_THREADS, (R == 4 && sizeof(T) == 8) ? 2 : WENO5_MINB)
weno_xz_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* __restrict__ W, const T* Un, T* Uout, Ctl* ctl,
               int zc) {
    using S = WenoXZShape<T, R>;
    using Win = typename S::Win;
    constexpr int M = 2 * R, NV = S::NV, NS = S::NS, NH = S::NH, NHL = S::NHL, RWX = S::RWX, D = WENO_DEPTH;
    constexpr int TH = WENO_THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);
    const int lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32 + lane;
    const int i0 = (int)blockIdx.x * 31 - 1, i = i0 + lane;
    const int j = (int)blockIdx.y * WENO_ROWS + wy;
    if (j >= G.n[1]) return;   // whole warp
    T* row = sm + D * S::STAGE + wy * NH * RWX;            // [NH][RWX], this warp's
    T* park = sm + D * S::STAGE + WENO_ROWS * NH * RWX + tid; // [NF][TH]: this thread's last z-flux
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

    auto issue = [&](int k) {
        if (k < k1) {
            T* st = sm + ((k - k0) % D) * S::STAGE;
            T* dst = st + tid;
            const long long q = p0 + (long long)(k - k0) * G.sxy, qr = q + (long long)R * G.sxy;
#pragma unroll
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + c * TH, Us + c * G.fs + qr);
            cp_async<sizeof(T)>(dst + (NF + 0) * TH, W + (W_V + 2) * G.fs + qr);
            cp_async<sizeof(T)>(dst + (NF + 1) * TH, W + W_P * G.fs + qr);
            cp_async<sizeof(T)>(dst + (NF + 2) * TH, W + (W_AX + 2) * G.fs + qr);
            cp_async<sizeof(T)>(dst + (NV + 0) * TH, W + (W_V + 0) * G.fs + q);
            cp_async<sizeof(T)>(dst + (NV + 1) * TH, W + (W_AX + 0) * G.fs + q);
            if (use_un) {
#pragma unroll
                for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + (NV + 2 + c) * TH, Un + c * G.fs + q);
            }
            if (lane < NHL) {
                T* hd = st + NS * TH + (wy * NHL + lane) * NH;
                const long long qh = ph + (long long)(k - k0) * G.sxy;
#pragma unroll
                for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(hd + c, Us + c * G.fs + qh);
                cp_async<sizeof(T)>(hd + NF + 0, W + (W_V + 0) * G.fs + qh);
                cp_async<sizeof(T)>(hd + NF + 1, W + W_P * G.fs + qh);
                cp_async<sizeof(T)>(hd + NF + 2, W + (W_AX + 0) * G.fs + qh);
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d < D; ++d) issue(k0 + d);

    Win zw;
    T nxt[NV];
#pragma unroll
    for (int m = 0; m < M; ++m) {   // cells k0-R .. k0+R-1
        Win::fetch(nxt, Us, W, G.fs, p0 + (long long)(m - R) * G.sxy);
        if (m == 0) zw.first(nxt);
        else zw.put(m, nxt);
    }
    const T eps = (T)A.eps;
    {
        T f0[NF];
        llf_weno_iface2<T, R, 2>(zw, eps, f0);   // face k0 - 1/2
#pragma unroll
        for (int c = 0; c < NF; ++c) park[c * TH] = f0[c];
    }
    // the interface function returns twice the flux: the 1/2 of the Lax-Friedrichs split goes into dt/dx
    const T dtdx = (T)(A.mode == 1 ? 0.5 * A.inv_dx : 0.5 * ctl->dt * A.inv_dx), ca = (T)A.ca, cb = (T)A.cb;

    for (int k = k0; k < k1; ++k) {
        cp_async_wait<D - 1>();   // plane k's stage has landed
        const T* st = sm + ((k - k0) % D) * S::STAGE;
        const T* src = st + tid;
#pragma unroll
        for (int v = 0; v < NV; ++v) nxt[v] = src[v * TH];
        zw.shift();
        zw.put(M - 1, nxt);
        __syncwarp();             // every lane is done with the row of plane k-1
#pragma unroll
        for (int c = 0; c < NF; ++c) row[c * RWX + lane + R - 1] = zw.uu[c][R - 1];
        row[(NF + 0) * RWX + lane + R - 1] = src[NV * TH];
        row[(NF + 1) * RWX + lane + R - 1] = zw.ww[1][R - 1];
        row[(NF + 2) * RWX + lane + R - 1] = src[(NV + 1) * TH];
        if (lane < NHL) {   // the halo cells go from their slots straight into the row
            const T* hs = st + NS * TH + (wy * NHL + lane) * NH;
#pragma unroll
            for (int a = 0; a < NH; ++a) row[a * RWX + hq] = hs[a];
        }
        __syncwarp();
        T L[NF], f[NF];
        llf_weno_iface2<T, R, 2>(zw, eps, f);
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            L[c] = park[c * TH] - f[c];
            park[c * TH] = f[c];
        }
#pragma unroll
        for (int c = 0; c < NF; ++c) f[c] = (T)0;
        if (need_x) {
            XRowAcc<T> acc{row + lane, RWX};
            llf_weno_iface2<T, R, 0>(acc, eps, f);
        }
#pragma unroll
        for (int c = 0; c < NF; ++c) L[c] += shfl_up1<T>(f[c]) - f[c];
        if (own) {
            const long long q = p0 + (long long)(k - k0) * G.sxy;
            if (A.mode == 1) {
#pragma unroll
                for (int c = 0; c < NF; ++c) Uout[c * G.fs + q] = L[c] * dtdx;
            } else {
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    T v = tfma(dtdx, L[c], zw.uu[c][R - 1]);
                    if (use_un) v = tfma(ca, src[(NV + 2 + c) * TH], cb * v);   // u^n: read late, it is only needed here
                    Uout[c * G.fs + q] = v;
                }
            }
        }
        issue(k + D);             // refill the slot just consumed
    }
}

// ---------------------------------------------------------------------------------------------------------
template <class T, int R>
constexpr size_t weno_y_smem_bytes() {
    return sizeof(T) * ((size_t)WENO_DEPTH * (NF + 3 + NF) + NF) * WENO_THREADS;
}

template <class T, int R, bool EPI>
__global__ void __launch_bounds__(WENO_THREADS, (R == 4 && sizeof(T) == 8) ? 2 : WENO5_MINB)
weno_y_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* __restrict__ W, T* Uout, T* Wnext, Ctl* ctl,
              int yc) {
    using Win = WenoWindow<T, R, 1>;
    constexpr int M = 2 * R, NV = Win::NV, NVO = NV + NF, D = WENO_DEPTH, TH = WENO_THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);   // [D][NVO][TH], then [NF][TH]
    const int tid = threadIdx.x + 32 * threadIdx.y;
    // the last flux is needed once per cell of the march: parked in shared memory, the kernel fits its register
    // budget without spilling
    T* park = sm + D * NVO * TH + tid;
    const int i = blockIdx.x * 32 + threadIdx.x;
    const int kz = blockIdx.y * WENO_ROWS + threadIdx.y;
    // lanes beyond the grid leave; the ballot (taken while the warp is whole) is the mask of the final reduction
    const unsigned wmask = __ballot_sync(0xffffffffu, i < G.n[0] && kz < G.n[2]);
    if (i >= G.n[0] || kz >= G.n[2]) return;
    const long long ms = G.sx;
    const int j0 = (int)blockIdx.z * yc;
    const int j1 = min(j0 + yc, G.n[1]);
    const long long p0 = G.pidx(i, j0, kz);
    auto issue = [&](int j) {   // window cell j+R and the old output of cell j
        if (j < j1) {
            T* dst = sm + ((j - j0) % D) * NVO * TH + tid;
            const long long q = p0 + (long long)(j - j0) * ms;
            const long long qr = q + (long long)R * ms;
#pragma unroll
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + c * TH, Us + c * G.fs + qr);
            cp_async<sizeof(T)>(dst + (NF + 0) * TH, W + (W_V + 1) * G.fs + qr);
            cp_async<sizeof(T)>(dst + (NF + 1) * TH, W + W_P * G.fs + qr);
            cp_async<sizeof(T)>(dst + (NF + 2) * TH, W + (W_AX + 1) * G.fs + qr);
#pragma unroll
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + (NV + c) * TH, Uout + c * G.fs + q);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d < D; ++d) issue(j0 + d);

    Win yw;
    T nxt[NV];
#pragma unroll
    for (int m = 0; m < M; ++m) {
        Win::fetch(nxt, Us, W, G.fs, p0 + (long long)(m - R) * ms);
        if (m == 0) yw.first(nxt);
        else yw.put(m, nxt);
    }
    const T eps = (T)A.eps;
    {
        T f0[NF];
        llf_weno_iface2<T, R, 1>(yw, eps, f0);
#pragma unroll
        for (int c = 0; c < NF; ++c) park[c * TH] = f0[c];
    }
    const T coef = A.mode == 1 ? (T)(0.5 * A.inv_dx) : (T)(0.5 * A.cb * ctl->dt * A.inv_dx);   // twice the flux comes in
    int flag = 0;
    double amax = 0.0;
    for (int j = j0; j < j1; ++j) {
        T f[NF], o[NF];
        cp_async_wait<D - 1>();   // the oldest stage (cell j) has landed
        const T* src = sm + ((j - j0) % D) * NVO * TH + tid;
#pragma unroll
        for (int v = 0; v < NV; ++v) nxt[v] = src[v * TH];
        yw.shift();
        yw.put(M - 1, nxt);
        llf_weno_iface2<T, R, 1>(yw, eps, f);
        const long long q = p0 + (long long)(j - j0) * ms;
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            o[c] = tfma(coef, park[c * TH] - f[c], src[(NV + c) * TH]);   // old output: read late
            Uout[c * G.fs + q] = o[c];
            park[c * TH] = f[c];
        }
        issue(j + D);             // refill the slot just consumed
        if (EPI) {
            T w[NW];
            int fl = 0;
            prim_of_cell(o, w, fl, A.eos);
#pragma unroll
            for (int a = 0; a < NW; ++a) Wnext[a * G.fs + q] = w[a];
            if (A.epi_max) amax = fmax(amax, fmax((double)w[W_AX], fmax((double)w[W_AX + 1], (double)w[W_AX + 2])));
            flag |= fl;
        }
    }
    if (EPI && A.epi_max) warp_max_to(amax, &ctl->maxspeed_next_bits, wmask);   // all three axes are active here
    if (flag) ctl->flag = 1;
}

template <class T, int R>
int configure_weno(char* err, size_t errlen) {
    cudaError_t e = cudaFuncSetAttribute(weno_xz_kernel<T, R>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)WenoXZShape<T, R>::smem_bytes());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(weno_y_kernel<T, R, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)weno_y_smem_bytes<T, R>());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(weno_y_kernel<T, R, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)weno_y_smem_bytes<T, R>());
    if (e != cudaSuccess) {
        snprintf(err, errlen, "cudaFuncSetAttribute (weno): %s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

// stage = x/z kernel (writes Uout) + y sweep (adds L_y; epilogue -> Wnext, and the CFL max in stage 3)
template <class T, int R>
int launch_weno(const Geom& G, const StageArgs& A, const T* Us, const T* W, const T* Un, T* Uout, T* Wnext, Ctl* ctl,
                int zc, int yc, cudaStream_t st, int* launches, char* err, size_t errlen) {
    const dim3 b(32, WENO_ROWS, 1);
    const dim3 g((G.n[0] + 30) / 31, (G.n[1] + WENO_ROWS - 1) / WENO_ROWS, (G.n[2] + zc - 1) / zc);
    weno_xz_kernel<T, R><<<g, b, WenoXZShape<T, R>::smem_bytes(), st>>>(G, A, Us, W, Un, Uout, ctl, zc);
    const dim3 gy((G.n[0] + 31) / 32, (G.n[2] + WENO_ROWS - 1) / WENO_ROWS, (G.n[1] + yc - 1) / yc);
    if (Wnext != nullptr && A.mode != 1)
        weno_y_kernel<T, R, true><<<gy, b, weno_y_smem_bytes<T, R>(), st>>>(G, A, Us, W, Uout, Wnext, ctl, yc);
    else
        weno_y_kernel<T, R, false><<<gy, b, weno_y_smem_bytes<T, R>(), st>>>(G, A, Us, W, Uout, nullptr, ctl, yc);
    *launches = 2;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(err, errlen, "%s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

}  // namespace hydro
