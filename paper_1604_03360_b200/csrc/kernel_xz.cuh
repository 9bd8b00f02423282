// kernel_xz.cuh -- x and z fluxes of one Runge-Kutta stage in ONE marching kernel without block barriers
// (stage layout "xz + y").
//
// A warp is a row of 32 consecutive x positions (lane 0 is the helper column one cell below the 31 cells the
// warp owns), a block is four such rows, and every thread marches along z through a chunk of planes:
//   z: the 2r-cell stencil of the thread's column lives in a register window (as in the marching sweep);
//   x: the plane-k cells of the window are exactly the row the x-stencil needs, so every lane writes its own
//      (conserved, winv, p, a_x) into a per-WARP shared-memory row, 2r-1 halo lanes add the cells beyond the
//      row's ends, and after a __syncwarp each lane reads its 2r-cell x-stencil from that row.  The lower-face
//      flux comes from lane-1 by shuffle.
// Every global read of the loop (window cell k+r, a_x and u^n of plane k, the halo columns of plane k) is a
// cp.async into the thread's own slots XZ_DEPTH planes ahead.  Warps never wait for one another: the only
// synchronisation is __syncwarp around the row.  Writes Uout = ca u^n + cb (u_s + dt (L_x + L_z)); the y sweep
// (z_sweep_kernel<..., DIR = 1>) then adds L_y and runs the con2prim epilogue.
#pragma once
#include "kernel_fused.cuh"

namespace hydro {

constexpr int XZ_DEPTH = 3;
constexpr int XZ_ROWS = 4;   // warps per block

template <class T, int SCHEME>
struct XZShape {
    using Win = ZWindow<T, SCHEME, 2>;
    static constexpr int R = Win::R;
    static constexpr int NV = Win::NV;                        // window cell: conserved (+ winv, p, a_z)
    static constexpr int NAX = SCHEME == 2 ? 0 : 1;           // a_x of plane k
    static constexpr int NS = NV + NAX + NF;                  // + u^n of plane k: slots per thread and stage
    static constexpr int NH = SCHEME == 2 ? NF : NF + 3;      // row arrays: conserved (+ winv, p, a_x)
    static constexpr int NHL = 2 * R - 1;                     // halo lanes: R-1 cells below, R cells above the row
    static constexpr int RWX = 32 + 2 * R - 1;                // cells of a row with halo
    static constexpr int STAGE = NS * 32 * XZ_ROWS + XZ_ROWS * NHL * NH;
    // pipeline stages, the warps' rows, and one parking slot per thread and field for the last z-flux (it is
    // only needed once per plane; parked, the kernel fits its register budget without spilling)
    static constexpr size_t smem_bytes() {
        return sizeof(T) * ((size_t)XZ_DEPTH * STAGE + XZ_ROWS * NH * RWX + NF * 32 * XZ_ROWS);
    }
};

template <class T, int SCHEME>
__global__ void __launch_bounds__(32 * XZ_ROWS, (SCHEME == 1 && sizeof(T) == 8) ? 2 : 3)
xz_sweep_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* __restrict__ W, const T* Un,
                T* Uout, Ctl* ctl, int zc) {
    using S = XZShape<T, SCHEME>;
    using Win = typename S::Win;
    constexpr int R = S::R, M = 2 * R, NV = S::NV, NS = S::NS, NH = S::NH, NHL = S::NHL, RWX = S::RWX, D = XZ_DEPTH;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);
    const int lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32 + lane;
    const int i0 = (int)blockIdx.x * 31 - 1, i = i0 + lane;
    const int j = (int)blockIdx.y * XZ_ROWS + wy;
    if (j >= G.n[1]) return;   // whole warp
    T* row = sm + D * S::STAGE + wy * NH * RWX;            // [NH][RWX], this warp's
    T* park = sm + D * S::STAGE + XZ_ROWS * NH * RWX + tid; // [NF][128]: this thread's last z-flux
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
            for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + c * 128, Us + c * G.fs + qr);
            if (SCHEME != 2) {
                cp_async<sizeof(T)>(dst + (NF + 0) * 128, W + W_INV * G.fs + qr);
                cp_async<sizeof(T)>(dst + (NF + 1) * 128, W + W_P * G.fs + qr);
                cp_async<sizeof(T)>(dst + (NF + 2) * 128, W + (W_AX + 2) * G.fs + qr);
                cp_async<sizeof(T)>(dst + NV * 128, W + (W_AX + 0) * G.fs + q);
            }
            if (use_un) {
#pragma unroll
                for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(dst + (NV + S::NAX + c) * 128, Un + c * G.fs + q);
            }
            if (lane < NHL) {
                T* hd = st + NS * 128 + (wy * NHL + lane) * NH;
                const long long qh = ph + (long long)(k - k0) * G.sxy;
#pragma unroll
                for (int c = 0; c < NF; ++c) cp_async<sizeof(T)>(hd + c, Us + c * G.fs + qh);
                if (SCHEME != 2) {
                    cp_async<sizeof(T)>(hd + NF + 0, W + W_INV * G.fs + qh);
                    cp_async<sizeof(T)>(hd + NF + 1, W + W_P * G.fs + qh);
                    cp_async<sizeof(T)>(hd + NF + 2, W + (W_AX + 0) * G.fs + qh);
                }
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
        zw.put(m, nxt);
    }
    // the helper lane and the idle lanes of a ragged last tile march through x-ghost columns, whose z-ghost cells
    // are edge ghosts nobody fills: their z-fluxes are discarded, and so must be their unphysical-state flag
    int zflag = 0;
    {
        T f0[NF];
        iface_from<T, SCHEME, 2>(zw, A, f0, zflag);   // face k0 - 1/2
#pragma unroll
        for (int c = 0; c < NF; ++c) park[c * 128] = f0[c];
    }
    const T dt = (T)ctl->dt, ca = (T)A.ca, cb = (T)A.cb, inv_dx = (T)A.inv_dx;

    for (int k = k0; k < k1; ++k) {
        cp_async_wait<D - 1>();   // plane k's stage has landed
        const T* st = sm + ((k - k0) % D) * S::STAGE;
        const T* src = st + tid;
        T axk = (T)0, hv[NH];
#pragma unroll
        for (int v = 0; v < NV; ++v) nxt[v] = src[v * 128];
        if (SCHEME != 2) axk = src[NV * 128];
        if (lane < NHL) {
            const T* hs = st + NS * 128 + (wy * NHL + lane) * NH;
#pragma unroll
            for (int a = 0; a < NH; ++a) hv[a] = hs[a];
        }
        zw.shift();
        zw.put(M - 1, nxt);
        __syncwarp();             // every lane is done with the row of plane k-1
#pragma unroll
        for (int c = 0; c < NF; ++c) row[c * RWX + lane + R - 1] = zw.uu[c][R - 1];
        if (SCHEME != 2) {
            row[(NF + 0) * RWX + lane + R - 1] = zw.ww[0][R - 1];
            row[(NF + 1) * RWX + lane + R - 1] = zw.ww[1][R - 1];
            row[(NF + 2) * RWX + lane + R - 1] = axk;
        }
        if (lane < NHL) {
#pragma unroll
            for (int a = 0; a < NH; ++a) row[a * RWX + hq] = hv[a];
        }
        __syncwarp();
        T L[NF], f[NF];
        iface_from<T, SCHEME, 2>(zw, A, f, zflag);
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            L[c] = park[c * 128] - f[c];
            park[c * 128] = f[c];
        }
#pragma unroll
        for (int c = 0; c < NF; ++c) f[c] = (T)0;
        if (need_x) {
            RectAcc<T> acc{row + lane, row + NF * RWX + lane, 1, RWX};
            iface_from<T, SCHEME, 0>(acc, A, f, flag);
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
                    if (use_un) v = tfma(ca, src[(NV + S::NAX + c) * 128], cb * v);   // u^n: read late, it is only needed here
                    Uout[c * G.fs + q] = v;
                }
            }
        }
        issue(k + D);             // refill the slot just consumed
    }
    if (flag || (own && zflag)) ctl->flag = 1;
}

template <class T, int SCHEME>
int configure_xz(FusedPlan& P) {
    cudaError_t e = cudaFuncSetAttribute(xz_sweep_kernel<T, SCHEME>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)XZShape<T, SCHEME>::smem_bytes());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(z_sweep_kernel<T, SCHEME, false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)zsweep_smem_bytes<T, SCHEME>());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(z_sweep_kernel<T, SCHEME, (SCHEME != 2), 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)zsweep_smem_bytes<T, SCHEME>());
    if (e != cudaSuccess) {
        snprintf(P.err, sizeof P.err, "cudaFuncSetAttribute (xz): %s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

// stage = xz sweep (writes Uout) + y sweep (adds L_y, con2prim epilogue)
template <class T, int SCHEME>
int launch_xz_y(FusedPlan& P, const Geom& G, const StageArgs& A, const T* Us, const T* W, const T* Un, T* Uout,
                T* Wnext, Ctl* ctl, cudaStream_t st, int* launches) {
    const dim3 b(32, XZ_ROWS, 1);
    const dim3 g((G.n[0] + 30) / 31, (G.n[1] + XZ_ROWS - 1) / XZ_ROWS, (G.n[2] + P.tile_zc - 1) / P.tile_zc);
    xz_sweep_kernel<T, SCHEME><<<g, b, XZShape<T, SCHEME>::smem_bytes(), st>>>(G, A, Us, W, Un, Uout, ctl, P.tile_zc);
    const dim3 by(32, 4, 1);
    const dim3 gy((G.n[0] + 31) / 32, (G.n[2] + 3) / 4, (G.n[1] + P.sweep_zc - 1) / P.sweep_zc);
    if (SCHEME != 2 && Wnext != nullptr)
        z_sweep_kernel<T, SCHEME, (SCHEME != 2), 1><<<gy, by, zsweep_smem_bytes<T, SCHEME>(), st>>>(G, A, Us, W, Uout, Wnext, ctl, P.sweep_zc);
    else
        z_sweep_kernel<T, SCHEME, false, 1><<<gy, by, zsweep_smem_bytes<T, SCHEME>(), st>>>(G, A, Us, W, Uout, nullptr, ctl, P.sweep_zc);
    *launches = 2;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(P.err, sizeof P.err, "%s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

}  // namespace hydro
