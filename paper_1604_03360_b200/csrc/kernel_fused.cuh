// kernel_fused.cuh -- stage kernels: L(u) of Eq. (2) fused with the SSP-RK3 combination
// (a9), every interface flux computed once.  This header holds
//   * z_sweep_kernel<T, SCHEME, EPI, DIR>: the marching sweep along y (DIR = 1, default layout) or z (DIR = 2):
//     thread per (x, other axis) column, 2r-cell stencil in a register window, cp.async pipeline, optional
//     con2prim epilogue.  With kernel_xz.cuh's x/z marching kernel it forms the DEFAULT stage ("layout" 1);
//   * stage_tiled_kernel<T, SCHEME, WITH_Z>: the TMA-staged x/y tile kernel of the alternative layout
//     ("layout" 0: tile kernel, then the z sweep) and, with WITH_Z, the single-kernel variant ("split_z" 0);
//   * the plan (tensor maps, shared-memory attributes) and the launchers.
//
// stage_tiled_kernel<T, SCHEME, WITH_Z>
//   A block is 32 x TY threads over an (x, y) tile and marches along z through a chunk of planes.  Thread
//   (lane, ty) sits on cell (i0 + lane, j0 + ty), i0 = 31 bx - 1, j0 = (TY-1) by - 1: column lane = 0 and
//   row ty = 0 are helper positions one cell below the tile, the other 31 x (TY-1) positions own a cell.
//   Per plane the halo'd rectangle of the tile (conserved fields, winv, p, a_x, a_y; R-1 / R cells of halo)
//   is brought into shared memory by TMA (two cp.async.bulk.tensor boxes per plane, issued by one thread and
//   awaited on an mbarrier), double buffered one plane ahead, and a thread computes
//   only UPPER-face fluxes from it:
//     x: f(i+1/2) by every thread of an owning row     -> lower face from lane-1 by warp shuffle
//     y: f(j+1/2) by every thread of an owning column  -> lower face from row ty-1 through shared memory
//   WITH_Z: z: f(k+1/2) by owning threads from a register window of the column (cells k-R+1 .. k+R,
//     shifted and refilled by one prefetched plane per step) -> lower face is last plane's flux.
//   Redundant work: one column of x-fluxes per 31, one row of y-fluxes per TY-1, one z-flux per chunk.
#pragma once
#include <cuda.h>

#include <cstdio>
#include <cstring>

#include "grid.cuh"
#include "kernel_generic.cuh"
#include "kernels_aux.cuh"

namespace hydro {

constexpr int FUSED_ZC = 64;    // default planes per z-chunk of the tiled kernel ("tile_zc" option)
constexpr int ZSWEEP_ZC = 128;  // default planes per z-chunk of the z sweep ("sweep_zc" option)

struct FusedPlan {
    int split_z = 1;  // 1: x/y tiled kernel + z sweep kernel; 0: one kernel with the z window inside
    int tile_zc = FUSED_ZC, sweep_zc = ZSWEEP_ZC;
    int layout = 1;   // split stage: 1 = x/z marching kernel + y sweep (default), 0 = x/y tile kernel + z sweep
    // TMA descriptors of the three padded state buffers and of the primitive arrays: 4-D tensors
    // (x, y, z, array) with box (RW, RH, 1, 5 or 4); one set per kernel variant [split, with z] because the
    // tile height differs
    CUtensorMap mapU[2][3], mapW[2][2];
    const void* baseU[3] = {nullptr, nullptr, nullptr};
    const void* baseW[2] = {nullptr, nullptr};
    char err[256] = {0};
};

inline bool fused_supported(const Geom& G, int /*scheme*/, int /*precision*/) {
    return G.g[0] > 0 && G.g[1] > 0 && G.g[2] > 0;
}

template <class T>
__device__ __forceinline__ T shfl_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// z-stencil of one column held in registers while the block marches along z: cells k-R+1 .. k+R, per cell
// the five conserved fields and (WENO only) winv, p, a_z.  All indices are compile-time constants after
// unrolling, so the arrays live in registers.
template <class T, int SCHEME, int DIR = 2>
struct ZWindow {
    static constexpr int R = SCHEME == 0 ? 3 : (SCHEME == 1 ? 4 : 2);
    static constexpr int M = 2 * R;
    static constexpr int NWZ = SCHEME == 2 ? 0 : 3;  // winv, p, a_z
    static constexpr int NV = NF + NWZ;
    T uu[NF][M];
    T ww[NWZ > 0 ? NWZ : 1][M];
    __device__ __forceinline__ T u(int c, int k) const { return uu[c][k]; }
    __device__ __forceinline__ T w(int a, int k) const { return ww[a == W_INV ? 0 : (a == W_P ? 1 : 2)][k]; }
    // values of one cell, fetched ahead of use
    static __device__ __forceinline__ void fetch(T v[NV], const T* __restrict__ U, const T* __restrict__ W,
                                                 long long fs, long long q) {
#pragma unroll
        for (int c = 0; c < NF; ++c) v[c] = __ldg(U + c * fs + q);
        if (NWZ > 0) {
            v[NF + 0] = __ldg(W + W_INV * fs + q);
            v[NF + 1] = __ldg(W + W_P * fs + q);
            v[NF + 2] = __ldg(W + (W_AX + DIR) * fs + q);
        }
    }
    __device__ __forceinline__ void put(int m, const T v[NV]) {
#pragma unroll
        for (int c = 0; c < NF; ++c) uu[c][m] = v[c];
#pragma unroll
        for (int a = 0; a < NWZ; ++a) ww[a][m] = v[NF + a];
    }
    __device__ __forceinline__ void shift() {
#pragma unroll
        for (int m = 0; m + 1 < M; ++m) {
#pragma unroll
            for (int c = 0; c < NF; ++c) uu[c][m] = uu[c][m + 1];
#pragma unroll
            for (int a = 0; a < NWZ; ++a) ww[a][m] = ww[a][m + 1];
        }
    }
};

template <class T, int SCHEME, int DIR, class Acc>
__device__ __forceinline__ void iface_from(const Acc& acc, const StageArgs& A, T fh[NF], int& flag) {
    constexpr int R = SCHEME == 0 ? 3 : (SCHEME == 1 ? 4 : 2);
    if constexpr (SCHEME == 2) musta_force_iface<T, DIR>(acc, A.musta_K, (T)A.musta_C, A.limiter, A.eos.kind, (T)A.eos.p0, fh, flag);
    else llf_weno_iface<T, R, DIR>(acc, (T)A.eps, fh);
}

// ---- TMA (cp.async.bulk.tensor) + mbarrier, raw PTX for sm_100a -------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra WAIT_LOOP;\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// box of a 4-D tensor (x, y, z, array) -> shared memory; out-of-bounds parts of the box are zero-filled
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3,
                                            unsigned long long* bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
        : "memory");
}

// stencil accessor into the shared-memory rectangle of one plane: conserved arrays at ub, (winv, p, a_x, a_y)
// at wb, array stride astride, stencil stride `stride` (1 along x, the row pitch along y)
template <class T>
struct RectAcc {
    const T* ub;
    const T* wb;
    int stride, astride;
    __device__ __forceinline__ T u(int c, int k) const { return ub[c * astride + k * stride]; }
    __device__ __forceinline__ T w(int a, int k) const { return wb[a * astride + k * stride]; }
};

template <class T, int SCHEME, bool WITH_Z>
struct TileShape {
    static constexpr int R = SCHEME == 0 ? 3 : (SCHEME == 1 ? 4 : 2);
    // rows per block (one of them the helper row).  16 rows (512 threads, one block per SM) halve the redundant
    // y-fluxes but measured slower than two independent 256-thread blocks per SM (18.1 vs 17.2 ms per stage,
    // WENO5 fp64 512^3): one barrier then stalls the whole SM.
    static constexpr int TY = 8;
    // resident blocks per SM the register budget is sized for: fp64 WENO5/MUSTA 2 (128 registers), fp64 WENO7
    // and the variant with the z window inside 1, fp32 WENO5/MUSTA 3 (80 registers suffice; left free the
    // compiler takes 126 and the fp32 step is 25 % slower)
    static constexpr int MIN_BLOCKS = (TY == 16 || WITH_Z || (SCHEME == 1 && sizeof(T) == 8)) ? 1
                                      : (sizeof(T) == 4 && SCHEME != 1) ? 3 : 2;
    static constexpr int Q = 16 / (int)sizeof(T);                       // elements per 16 bytes
    // box width (x): 32 + 2R - 1 cells plus up to Q-1 of lead-in, because TMA wants the box to start on a
    // 16-byte boundary of the row and to be a multiple of 16 bytes wide
    static constexpr int RW = (32 + 2 * R - 1 + (Q - 1) + Q - 1) / Q * Q;
    static constexpr int RH = TY + 2 * R - 1;                     // box height (y)
    static constexpr int NWA = SCHEME == 2 ? 0 : 4;                     // winv, p, a_x, a_y
    static constexpr int CELLS = RW * RH;
    static constexpr int U_ELEMS = (NF * CELLS * (int)sizeof(T) + 127) / 128 * 128 / (int)sizeof(T);
    static constexpr int W_ELEMS = (NWA * CELLS * (int)sizeof(T) + 127) / 128 * 128 / (int)sizeof(T);
    static constexpr int BUF_ELEMS = U_ELEMS + W_ELEMS;
    static constexpr unsigned TX_BYTES = (unsigned)((NF + NWA) * CELLS * sizeof(T));
    static constexpr size_t smem_bytes() {
        return sizeof(T) * (2 * (size_t)BUF_ELEMS + 2 * TY * NF * 32) + 2 * sizeof(unsigned long long);
    }
};

template <class T, int SCHEME, bool WITH_Z>
__global__ void __launch_bounds__(32 * TileShape<T, SCHEME, WITH_Z>::TY, TileShape<T, SCHEME, WITH_Z>::MIN_BLOCKS)
stage_tiled_kernel(const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapW, Geom G,
                   StageArgs A, const T* __restrict__ Us, const T* __restrict__ W, const T* Un, T* Uout, Ctl* ctl,
                   int zc) {
    using S = TileShape<T, SCHEME, WITH_Z>;
    constexpr int R = S::R, M = 2 * R, FUSED_TY = S::TY;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    T* rect = reinterpret_cast<T*>(smem_raw);                                  // [2][BUF_ELEMS]
    T* fy_s = rect + 2 * S::BUF_ELEMS;                                         // [2][TY][NF][32]
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(fy_s + 2 * FUSED_TY * NF * 32);
    const int lane = threadIdx.x, ty = threadIdx.y;
    const bool leader = lane == 0 && ty == 0;
    const int i0 = (int)blockIdx.x * 31 - 1, j0 = (int)blockIdx.y * (FUSED_TY - 1) - 1;
    const int i = i0 + lane, j = j0 + ty;
    const int k0 = (int)blockIdx.z * zc;
    const int k1 = min(k0 + zc, G.n[2]);
    const bool row_ok = ty >= 1 && j < G.n[1];
    const bool col_ok = lane >= 1 && i < G.n[0];
    const bool own = row_ok && col_ok;
    const bool need_x = row_ok && i < G.n[0];  // i >= -1 always
    const bool need_y = col_ok && j < G.n[1];  // j >= -1 always
    const int x_first = i0 - R + 1 + G.g[0], y_lo_pad = j0 - R + 1 + G.g[1];
    const int x_lo_pad = x_first & ~(S::Q - 1);   // 16-byte aligned start of the box
    const int xo = x_first - x_lo_pad + lane;      // this thread's first stencil column inside the box
    const int ic = min(i, G.n[0] - 1), jc = min(j, G.n[1] - 1);
    long long p = G.pidx(ic, jc, k0);
    int flag = 0;
    const T inv_dx = (T)A.inv_dx;

    if (leader) {
        mbar_init(&bars[0], 1);
        mbar_init(&bars[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (leader) {   // plane k0 -> buffer 0
        mbar_expect_tx(&bars[0], S::TX_BYTES);
        tma_load_4d(rect, &mapU, x_lo_pad, y_lo_pad, k0 + G.g[2], 0, &bars[0]);
        if (S::NWA > 0) tma_load_4d(rect + S::U_ELEMS, &mapW, x_lo_pad, y_lo_pad, k0 + G.g[2], 0, &bars[0]);
    }

    T fz_lo[NF];
    ZWindow<T, SCHEME> zw;
    T nxt[ZWindow<T, SCHEME>::NV];
    if (WITH_Z && own) {
#pragma unroll
        for (int m = 0; m < M; ++m) {  // cells k0-R .. k0+R-1
            ZWindow<T, SCHEME>::fetch(nxt, Us, W, G.fs, p + (long long)(m - R) * G.sxy);
            zw.put(m, nxt);
        }
        iface_from<T, SCHEME, 2>(zw, A, fz_lo, flag);  // face k0 - 1/2
        ZWindow<T, SCHEME>::fetch(nxt, Us, W, G.fs, p + (long long)R * G.sxy);  // cell k0 + R
    }
    const T dt = (T)ctl->dt, ca = (T)A.ca, cb = (T)A.cb;

    for (int k = k0; k < k1; ++k, p += G.sxy) {
        const int b = (k - k0) & 1;
        // plane k+1 -> the other buffer; every thread finished reading it before last plane's barrier
        if (leader && k + 1 < k1) {
            T* dst = rect + (b ^ 1) * S::BUF_ELEMS;
            mbar_expect_tx(&bars[b ^ 1], S::TX_BYTES);
            tma_load_4d(dst, &mapU, x_lo_pad, y_lo_pad, k + 1 + G.g[2], 0, &bars[b ^ 1]);
            if (S::NWA > 0) tma_load_4d(dst + S::U_ELEMS, &mapW, x_lo_pad, y_lo_pad, k + 1 + G.g[2], 0, &bars[b ^ 1]);
        }
        const T* rb = rect + b * S::BUF_ELEMS;
        T L[NF] = {0, 0, 0, 0, 0}, us_c[NF] = {0, 0, 0, 0, 0};
        if (WITH_Z && own) {
            T f[NF];
            zw.shift();
            zw.put(M - 1, nxt);
            if (k + 1 < k1) ZWindow<T, SCHEME>::fetch(nxt, Us, W, G.fs, p + (long long)(R + 1) * G.sxy);
            iface_from<T, SCHEME, 2>(zw, A, f, flag);
#pragma unroll
            for (int c = 0; c < NF; ++c) {
                L[c] = fz_lo[c] - f[c];
                fz_lo[c] = f[c];
            }
        }
        mbar_wait(&bars[b], ((k - k0) >> 1) & 1);   // plane k has landed in rect[b]
        if (ty >= 1) {  // warp-uniform: the helper row has no x work
            T f[NF] = {0, 0, 0, 0, 0};
            if (need_x) {
                const int o = (ty + R - 1) * S::RW + xo;
                RectAcc<T> acc{rb + o, rb + S::U_ELEMS + o, 1, S::CELLS};
                iface_from<T, SCHEME, 0>(acc, A, f, flag);
            }
#pragma unroll
            for (int c = 0; c < NF; ++c) {
                const T lo = shfl_up1<T>(f[c]);
                if (own) L[c] += lo - f[c];
            }
        }
        {
            T f[NF] = {0, 0, 0, 0, 0};
            if (need_y) {
                const int o = ty * S::RW + xo + R - 1;
                RectAcc<T> acc{rb + o, rb + S::U_ELEMS + o, S::RW, S::CELLS};
                iface_from<T, SCHEME, 1>(acc, A, f, flag);
            }
            T* fy = fy_s + b * FUSED_TY * NF * 32;
#pragma unroll
            for (int c = 0; c < NF; ++c) fy[(ty * NF + c) * 32 + lane] = f[c];
            // own cell's stage value (centre of the rectangle), read before rect[b] may be refilled
            if (own && A.mode != 1) {
                const T* uc = rb + (ty + R - 1) * S::RW + xo + R - 1;
#pragma unroll
                for (int c = 0; c < NF; ++c) us_c[c] = uc[c * S::CELLS];
            }
            __syncthreads();  // y-fluxes visible; everyone is done reading rect[b]
            if (own) {
#pragma unroll
                for (int c = 0; c < NF; ++c) L[c] += fy[((ty - 1) * NF + c) * 32 + lane] - f[c];
            }
        }
        if (own) {
            if (A.mode == 1) {
#pragma unroll
                for (int c = 0; c < NF; ++c) Uout[c * G.fs + p] = L[c] * inv_dx;
            } else {
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    T v = tfma(dt, L[c] * inv_dx, us_c[c]);
                    if (A.ca != 0.0) v = tfma(ca, Un[c * G.fs + p], cb * v);
                    Uout[c * G.fs + p] = v;
                }
            }
        }
    }
    if (flag) ctl->flag = 1;
}

// ---- cp.async (LDGSTS) helpers: per-thread asynchronous global -> shared copies ---------------------
template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(smem_u32(smem)), "l"(gmem), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

constexpr int ZSWEEP_THREADS = 128;
constexpr int ZSWEEP_DEPTH = 3;   // planes in flight

// Marching sweep along axis DIR (2: z, 1: y): Uout += coef * (f(m-1/2) - f(m+1/2)), coef = cb dt / dx
// (Runge-Kutta mode) or 1 / dx (mode 1).  One thread per (x, other axis) column, threads of a warp along x (so
// every access is coalesced whichever axis is marched), the 2r-cell stencil in a register window.
// Every global read of the marching loop (the new window cell m+R and the old Uout of cell m) is a
// cp.async into the thread's own shared-memory slots, ZSWEEP_DEPTH cells ahead: no load latency is
// exposed and no thread reads another thread's slots, so there is no barrier.
// EPI (WENO schemes, Runge-Kutta mode): the thread holds the finished stage value of its cell, so it also makes
// the next stage's primitives W' = (winv, p, a_x, a_y, a_z) of that cell (a2-a3; written to the OTHER W buffer,
// this stage's W is still being read by neighbouring chunks) and, in stage 3, the max signal speed of the new
// state (a4): the separate con2prim pass over the grid disappears from the step.
template <class T, int SCHEME, bool EPI, int DIR = 2>
__global__ void __launch_bounds__(ZSWEEP_THREADS, (SCHEME == 1 && sizeof(T) == 8) ? 2 : 3)
z_sweep_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* __restrict__ W, T* Uout, T* Wnext, Ctl* ctl,
               int zc) {
    using Win = ZWindow<T, SCHEME, DIR>;
    constexpr int R = Win::R, M = 2 * R, NV = Win::NV, NWZ = Win::NWZ;
    constexpr int NVO = NV + NF, D = ZSWEEP_DEPTH;
    constexpr int OTHER = DIR == 2 ? 1 : 2;   // the axis blockIdx.y / threadIdx.y run over
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);   // [D][NVO][ZSWEEP_THREADS], then [NF][ZSWEEP_THREADS]
    const int tid = threadIdx.x + blockDim.x * threadIdx.y;
    // the last flux is needed once per cell of the march: parked in shared memory, the kernel fits its
    // register budget without spilling (spills cost 6 % of the step when they were there)
    T* park = sm + D * NVO * ZSWEEP_THREADS + tid;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= G.n[0] || j >= G.n[OTHER]) return;
    const long long ms = DIR == 2 ? G.sxy : G.sx;   // stride of the marched axis
    const int k0 = (int)blockIdx.z * zc;
    const int k1 = min(k0 + zc, G.n[DIR]);
    long long p = DIR == 2 ? G.pidx(i, j, k0) : G.pidx(i, k0, j);
    int flag = 0;
    // stage for cell k of the march: window cell k+R and the old output of cell k
    auto issue = [&](int k) {
        if (k < k1) {
            T* dst = sm + ((k - k0) % D) * NVO * ZSWEEP_THREADS + tid;
            const long long q = p + (long long)(k - k0) * ms;
            const long long qr = q + (long long)R * ms;
#pragma unroll
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + c * ZSWEEP_THREADS, Us + c * G.fs + qr);
            if (NWZ > 0) {
                cp_async<sizeof(T)>(dst + (NF + 0) * ZSWEEP_THREADS, W + W_INV * G.fs + qr);
                cp_async<sizeof(T)>(dst + (NF + 1) * ZSWEEP_THREADS, W + W_P * G.fs + qr);
                cp_async<sizeof(T)>(dst + (NF + 2) * ZSWEEP_THREADS, W + (W_AX + DIR) * G.fs + qr);
            }
#pragma unroll
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + (NV + c) * ZSWEEP_THREADS, Uout + c * G.fs + q);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d < D; ++d) issue(k0 + d);

    Win zw;
    T nxt[NV];
#pragma unroll
    for (int m = 0; m < M; ++m) {
        Win::fetch(nxt, Us, W, G.fs, p + (long long)(m - R) * ms);
        zw.put(m, nxt);
    }
    {
        T f0[NF];
        iface_from<T, SCHEME, DIR>(zw, A, f0, flag);
#pragma unroll
        for (int c = 0; c < NF; ++c) park[c * ZSWEEP_THREADS] = f0[c];
    }
    const T coef = A.mode == 1 ? (T)A.inv_dx : (T)(A.cb * ctl->dt * A.inv_dx);
    const long long p0 = p;
    double amax = 0.0;
    for (int k = k0; k < k1; ++k) {
        T f[NF], o[NF];
        cp_async_wait<D - 1>();   // the oldest stage (cell k) has landed
        const T* src = sm + ((k - k0) % D) * NVO * ZSWEEP_THREADS + tid;
#pragma unroll
        for (int v = 0; v < NV; ++v) nxt[v] = src[v * ZSWEEP_THREADS];
        zw.shift();
        zw.put(M - 1, nxt);
        iface_from<T, SCHEME, DIR>(zw, A, f, flag);
        const long long q = p0 + (long long)(k - k0) * ms;
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            o[c] = tfma(coef, park[c * ZSWEEP_THREADS] - f[c], src[(NV + c) * ZSWEEP_THREADS]);   // old output: read late
            Uout[c * G.fs + q] = o[c];
            park[c * ZSWEEP_THREADS] = f[c];
        }
        issue(k + D);             // refill the slot just consumed
        if (EPI) {
            T w[NW];
            prim_of_cell(o, w, flag, A.eos);
#pragma unroll
            for (int a = 0; a < NW; ++a) Wnext[a * G.fs + q] = w[a];
            if (A.epi_max) amax = fmax(amax, fmax((double)w[W_AX], fmax((double)w[W_AX + 1], (double)w[W_AX + 2])));
        }
    }
    if (EPI && A.epi_max) {   // all three axes are active whenever this kernel runs
        const unsigned mask = __activemask();
#pragma unroll
        for (int o2 = 16; o2 > 0; o2 >>= 1) {
            const double other = __shfl_xor_sync(mask, amax, o2);
            if ((mask >> ((threadIdx.x & 31) ^ o2)) & 1u) amax = fmax(amax, other);   // partner lane exists
        }
        if ((threadIdx.x & 31) == 0 && amax > 0.0)
            atomicMax(&ctl->maxspeed_next_bits, (unsigned long long)__double_as_longlong(amax));
    }
    if (flag) ctl->flag = 1;
}

template <class T, int SCHEME>
constexpr size_t zsweep_smem_bytes() {
    return sizeof(T) * ((size_t)ZSWEEP_DEPTH * (ZWindow<T, SCHEME>::NV + NF) + NF) * ZSWEEP_THREADS;
}

template <class T, int SCHEME>
int configure_xz(FusedPlan& P);
template <class T, int SCHEME>
int launch_xz_y(FusedPlan& P, const Geom& G, const StageArgs& A, const T* Us, const T* W, const T* Un, T* Uout,
                T* Wnext, Ctl* ctl, cudaStream_t st, int* launches);

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// the driver entry point is looked up through the runtime, so the library has no link-time dependency on libcuda
inline EncodeTiledFn encode_tiled_fn() {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
        return nullptr;
    return (EncodeTiledFn)fn;
}

template <class T, int SCHEME>
int configure_tiled(FusedPlan& P, const Geom& G, void* const U[3], void* const W[2]) {
    using S = TileShape<T, SCHEME, false>;
    using SZ = TileShape<T, SCHEME, true>;
    cudaError_t e = cudaFuncSetAttribute(stage_tiled_kernel<T, SCHEME, false>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::smem_bytes());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(stage_tiled_kernel<T, SCHEME, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)SZ::smem_bytes());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(z_sweep_kernel<T, SCHEME, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)zsweep_smem_bytes<T, SCHEME>());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(z_sweep_kernel<T, SCHEME, (SCHEME != 2)>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)zsweep_smem_bytes<T, SCHEME>());
    if (e != cudaSuccess) {
        snprintf(P.err, sizeof P.err, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
        return -1;
    }
    if (configure_xz<T, SCHEME>(P) != 0) return -1;
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) {
        snprintf(P.err, sizeof P.err, "cuTensorMapEncodeTiled not available");
        return -1;
    }
    const CUtensorMapDataType dt = sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const cuuint64_t strides[3] = {(cuuint64_t)G.sx * sizeof(T), (cuuint64_t)G.sxy * sizeof(T), (cuuint64_t)G.fs * sizeof(T)};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    for (int v = 0; v < 2; ++v) {
        const int RW = v == 0 ? S::RW : SZ::RW, RH = v == 0 ? S::RH : SZ::RH;
        for (int m = 0; m < 5; ++m) {   // three state buffers, two primitive buffers
            const int narr = m < 3 ? NF : S::NWA;
            if (narr == 0) {
                memset(&P.mapW[v][m - 3], 0, sizeof(CUtensorMap));
                continue;
            }
            const cuuint64_t dims[4] = {(cuuint64_t)G.sx, (cuuint64_t)G.np[1], (cuuint64_t)G.np[2], (cuuint64_t)narr};
            const cuuint32_t box[4] = {(cuuint32_t)RW, (cuuint32_t)RH, 1, (cuuint32_t)narr};
            CUtensorMap* map = m < 3 ? &P.mapU[v][m] : &P.mapW[v][m - 3];
            void* base = m < 3 ? U[m] : W[m - 3];
            const CUresult r = enc(map, dt, 4, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) {
                snprintf(P.err, sizeof P.err, "cuTensorMapEncodeTiled failed: %d", (int)r);
                return -1;
            }
            if (m < 3) P.baseU[m] = base;
            else P.baseW[m - 3] = base;
        }
    }
    return 0;
}

inline int build_fused_plan(FusedPlan& P, const Geom& G, int scheme, int precision, void* const U[3], void* const W[2]) {
    if (precision == 0) {
        return scheme == 0 ? configure_tiled<double, 0>(P, G, U, W)
                           : scheme == 1 ? configure_tiled<double, 1>(P, G, U, W) : configure_tiled<double, 2>(P, G, U, W);
    }
    return scheme == 0 ? configure_tiled<float, 0>(P, G, U, W)
                       : scheme == 1 ? configure_tiled<float, 1>(P, G, U, W) : configure_tiled<float, 2>(P, G, U, W);
}

template <class T, int SCHEME>
int launch_fused_scheme(FusedPlan& P, const Geom& G, const StageArgs& A, const T* Us, const T* W, const T* Un, T* Uout,
                        T* Wnext, Ctl* ctl, cudaStream_t st, int* launches) {
    int m = -1;
    for (int q = 0; q < 3; ++q)
        if (P.baseU[q] == (const void*)Us) m = q;
    const int mw = P.baseW[1] == (const void*)W ? 1 : 0;
    if (m < 0) {
        snprintf(P.err, sizeof P.err, "stage input is not one of the context's state buffers");
        return -1;
    }
    if (P.split_z && P.layout == 1) return launch_xz_y<T, SCHEME>(P, G, A, Us, W, Un, Uout, Wnext, ctl, st, launches);
    if (P.split_z) {
        using S = TileShape<T, SCHEME, false>;
        const dim3 b(32, S::TY, 1);
        const dim3 g((G.n[0] + 30) / 31, (G.n[1] + S::TY - 2) / (S::TY - 1), (G.n[2] + P.tile_zc - 1) / P.tile_zc);
        stage_tiled_kernel<T, SCHEME, false><<<g, b, S::smem_bytes(), st>>>(P.mapU[0][m], P.mapW[0][mw], G, A, Us, W, Un, Uout, ctl, P.tile_zc);
        const dim3 bz(32, 4, 1);
        const dim3 gz((G.n[0] + 31) / 32, (G.n[1] + 3) / 4, (G.n[2] + P.sweep_zc - 1) / P.sweep_zc);
        if (SCHEME != 2 && Wnext != nullptr)
            z_sweep_kernel<T, SCHEME, (SCHEME != 2)><<<gz, bz, zsweep_smem_bytes<T, SCHEME>(), st>>>(G, A, Us, W, Uout, Wnext, ctl, P.sweep_zc);
        else
            z_sweep_kernel<T, SCHEME, false><<<gz, bz, zsweep_smem_bytes<T, SCHEME>(), st>>>(G, A, Us, W, Uout, nullptr, ctl, P.sweep_zc);
        *launches = 2;
    } else {
        using S = TileShape<T, SCHEME, true>;
        const dim3 b(32, S::TY, 1);
        const dim3 g((G.n[0] + 30) / 31, (G.n[1] + S::TY - 2) / (S::TY - 1), (G.n[2] + P.tile_zc - 1) / P.tile_zc);
        stage_tiled_kernel<T, SCHEME, true><<<g, b, S::smem_bytes(), st>>>(P.mapU[1][m], P.mapW[1][mw], G, A, Us, W, Un, Uout, ctl, P.tile_zc);
        *launches = 1;
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(P.err, sizeof P.err, "%s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

template <class T>
int launch_fused(FusedPlan& P, const Geom& G, int scheme, const StageArgs& A, const T* Us, const T* W, const T* Un,
                 T* Uout, T* Wnext, Ctl* ctl, cudaStream_t st, int* launches) {
    switch (scheme) {
        case 0: return launch_fused_scheme<T, 0>(P, G, A, Us, W, Un, Uout, Wnext, ctl, st, launches);
        case 1: return launch_fused_scheme<T, 1>(P, G, A, Us, W, Un, Uout, Wnext, ctl, st, launches);
        default: return launch_fused_scheme<T, 2>(P, G, A, Us, W, Un, Uout, Wnext, ctl, st, launches);
    }
}

}  // namespace hydro
