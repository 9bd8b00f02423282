// kernel_generic.cuh -- the any-shape stage kernel: L(u) of Eq. (2) fused with the
// SSP-RK3 combination (a9), one thread per interior cell, stencils read straight from
// global memory through L1/L2.  It evaluates both faces of every cell, so every interface flux is
// computed twice; it exists for the shapes the fused kernel does not take (inactive axes such as the
// 400 x 1 x 1 shock tube, grids smaller than a tile) and as the in-library cross-check of the fused one.
#pragma once
#include "grid.cuh"
#include "iface.cuh"
#include "kernels_aux.cuh"

namespace hydro {

template <class T>
struct GlobalAcc {  // stencil cell k lives at base + k*stride; field c at + c*fs
    const T* ub;
    const T* wb;
    long long fs, stride;
    __device__ __forceinline__ T u(int c, int k) const { return __ldg(ub + c * fs + k * stride); }
    __device__ __forceinline__ T w(int a, int k) const { return __ldg(wb + a * fs + k * stride); }
    template <int DIR, int M>
    __device__ __forceinline__ T alpha() const { return alpha_of_cells<T, M, DIR>(*this); }
};

struct StageArgs {
    double ca, cb;      // out = ca * u^n + cb * (u_stage + dt * L)      (a9)
    int mode;           // 0: Runge-Kutta combine, 1: write L itself (hydro_eval_L)
    double inv_dx;
    double eps;         // WENO epsilon (Q5)
    int musta_K;        // Q8
    double musta_C;     // Q7
    int limiter;        // MUSCL slope limiter: 0 minmod (Q6), 1 van Leer, 2 MC, 3 superbee
    EosArgs eos;        // equation of state: kind 0 p = e/3 (Q2), 1 p = p0, 2 tabulated p(e)
    int epi_max;        // z-sweep epilogue: also reduce the max signal speed of the new state (stage 3)
    int kbeg, kend;     // marching x/z kernels: the planes [kbeg, kend) this launch covers (the whole grid by default;
                        // the slab path launches the planes that need no z ghost first)
};

// flux at interface (cell p) + 1/2 along DIR; p = padded index of the cell on the low side
template <class T, int SCHEME, int DIR>
__device__ __forceinline__ void iface_generic(const Geom& G, const StageArgs& A, const T* __restrict__ U,
                                              const T* __restrict__ W, long long p, T fh[NF], int& flag) {
    const long long stride = DIR == 0 ? 1 : (DIR == 1 ? G.sx : G.sxy);
    constexpr int R = SCHEME == 0 ? 3 : (SCHEME == 1 ? 4 : 2);
    GlobalAcc<T> acc{U + p - (R - 1) * stride, W + p - (R - 1) * stride, G.fs, stride};
    if constexpr (SCHEME == 2) musta_force_iface<T, DIR>(acc, A.musta_K, (T)A.musta_C, A.limiter, A.eos, fh, flag);
    else {
        llf_weno_iface2<T, R, DIR>(acc, (T)A.eps, fh);   // twice the flux
#pragma unroll
        for (int c = 0; c < NF; ++c) fh[c] *= (T)0.5;
    }
}

template <class T, int SCHEME, int DIR>
__device__ __forceinline__ void add_axis(const Geom& G, const StageArgs& A, const T* __restrict__ U,
                                         const T* __restrict__ W, long long p, T L[NF], int& flag) {
    const long long stride = DIR == 0 ? 1 : (DIR == 1 ? G.sx : G.sxy);
    T fm[NF], fp[NF];
    // the loop keeps one copy of the (large) interface body in the instruction stream
    for (int side = 0; side < 2; ++side) {
        T f[NF];
        iface_generic<T, SCHEME, DIR>(G, A, U, W, p - (1 - side) * stride, f, flag);
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            if (side == 0) fm[c] = f[c];
            else fp[c] = f[c];
        }
    }
#pragma unroll
    for (int c = 0; c < NF; ++c) L[c] += (fm[c] - fp[c]) * (T)A.inv_dx;
}

template <class T, int SCHEME>
__global__ void __launch_bounds__(128) stage_generic_kernel(Geom G, StageArgs A, const T* __restrict__ Us,
                                                            const T* __restrict__ W, const T* Un, T* Uout, Ctl* ctl) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= G.n[0] || j >= G.n[1]) return;
    const long long p = G.pidx(i, j, k);
    T L[NF] = {0, 0, 0, 0, 0};
    int flag = 0;
    if (G.g[0]) add_axis<T, SCHEME, 0>(G, A, Us, W, p, L, flag);
    if (G.g[1]) add_axis<T, SCHEME, 1>(G, A, Us, W, p, L, flag);
    if (G.g[2]) add_axis<T, SCHEME, 2>(G, A, Us, W, p, L, flag);
    if (flag) ctl->flag = 1;
    if (A.mode == 1) {
#pragma unroll
        for (int c = 0; c < NF; ++c) Uout[c * G.fs + p] = L[c];
        return;
    }
    const T dt = (T)ctl->dt, ca = (T)A.ca, cb = (T)A.cb;
#pragma unroll
    for (int c = 0; c < NF; ++c) {
        T v = tfma(dt, L[c], Us[c * G.fs + p]);
        if (A.ca != 0.0) v = tfma(ca, Un[c * G.fs + p], cb * v);
        Uout[c * G.fs + p] = v;
    }
}

}  // namespace hydro
