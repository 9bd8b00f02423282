// kernel_weno.cuh -- stage kernels of the WENO schemes: L(u) of Eq. (2) fused with
// the SSP-RK3 combination (a9), with con2prim + signal speeds of every cell made as it enters a stencil
// window (a2-a3) and, in stage 3, with the CFL max of the finished cells (a4); every interface flux computed once
// (DESIGN.md section 7).  The only arrays in HBM are the conserved states.
//
//   weno_xz_kernel<T, R>        x and z fluxes in ONE marching kernel without block barriers.  A warp is a row of 32
//       consecutive x positions (lane 0 is the helper column one cell below the 31 cells the warp owns), a block is
//       four such rows, and every thread marches along z through a chunk of planes:
//         z: the 2r-cell stencil of the thread's column lives in a register window (conserved fields, v_z, p, a_z);
//            the primitives of a cell are made once, when it enters the window R planes ahead, together with its
//            (v_x, a_x), which wait in a small per-thread shared-memory ring until the cell's plane is the row;
//         x: the plane-k cells of the window are exactly the row the x-stencil needs, so every lane writes its own
//            (conserved, v_x, p, a_x) into a per-WARP shared-memory row, 2r-1 halo lanes add the cells beyond the
//            row's ends (and make their primitives), and after a __syncwarp each lane reads its 2r-cell x-stencil
//            from that row.  The lower-face flux comes from lane-1 by shuffle.
//       Writes Uout = ca u^n + cb (u_s + dt (L_x + L_z)).
//   weno_y_kernel<T, R, EPI>    the marching sweep along y: thread per (x, z) column, threads of a warp along x (so
//       every access is coalesced), adds cb dt L_y to Uout.  EPI (stage 3 of a CFL step): the thread holds the
//       finished cell, so it also reduces the max signal speed of the new state (a4) for the next step's dt.
// Every global read of the marching loops is a cp.async into the thread's own slots DEPTH cells ahead (pipeline.cuh).
//
// Performance model of these kernels (measured with microbenchmarks and confirmed to a few per
// cent by the ncu instruction counts under profiles/): an fp64 warp-instruction holds its scheduler's issue port for 2
// cycles, one with three distinct non-reused register operands for 3, and every other instruction adds about one
// more cycle: the kernels are bound by their total instruction count, not by occupancy.
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

// Primitives of one cell for the sweeps along the NDIR axes `dirs` (a2-a3): v_d, a_d per axis and p.  Made when a
// cell ENTERS a stencil window, from its conserved values alone: no primitive arrays exist in HBM (a stored v, p, a
// per cell and axis cost 120 B of DRAM traffic per cell and stage against ~50 fp64 instructions to make them again;
// the kernels are bound by instruction issue AND run at the board's power cap, where the bytes cost more clock than
// the flops).
// EOS: the closure is a compile-time constant of the kernel (0: p = e/3, 1: p = p0, 2: tabulated): a run-time branch here costs
// ~90 register moves per cell where its two sides merge.
template <class T, int NDIR, int EOS>
__device__ __forceinline__ void cell_prims(const T u[NF], const EosArgs& eos, const int (&dirs)[NDIR], T v[NDIR],
                                           T a[NDIR], T& p, int& flag) {
    T winv, v2;
    if (EOS == 1) {
        con2prim_p0(u[0], u[1], u[2], u[3], (T)eos.p0, winv, p, v2, flag);
#pragma unroll
        for (int d = 0; d < NDIR; ++d) {
            v[d] = u[1 + dirs[d]] * winv;
            a[d] = tabs(v[d]);
        }
    } else if (EOS == 2) {
        T cs2;
        con2prim_tab(u[0], u[1], u[2], u[3], eos, winv, p, v2, cs2, flag);
#pragma unroll
        for (int d = 0; d < NDIR; ++d) {
            v[d] = u[1 + dirs[d]] * winv;
            a[d] = signal_speed_cs(v[d], v2, cs2);
        }
    } else {
        con2prim(u[0], u[1], u[2], u[3], winv, p, v2, flag);
        const T id = speed_inv_den(v2);
#pragma unroll
        for (int d = 0; d < NDIR; ++d) {
            v[d] = u[1 + dirs[d]] * winv;
            a[d] = signal_speed(v[d], v2, id);
        }
    }
}

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
    // v = conserved fields, v_DIR, p, a_DIR of the cell
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
    static constexpr int NS = NF + NF;                        // pipeline slot: conserved of cell k+R, u^n of plane k
    static constexpr int NH = NF + 3;                         // row arrays: conserved, v_x, p, a_x
    static constexpr int NHL = 2 * R - 1;                     // halo lanes: R-1 cells below, R cells above the row
    static constexpr int RWX = 32 + 2 * R - 1;                // cells of a row with halo
    static constexpr int STAGE = NS * WENO_THREADS + WENO_ROWS * NHL * NF;
    static constexpr int RING = R + 1;                        // (v_x, a_x) of a cell wait R planes for their row
    // pipeline stages, the warps' rows, one parking slot per thread and field for the last z-flux (it is only
    // needed once per plane; parked, the kernel fits its register budget without spilling), the (v_x, a_x) ring
    static constexpr size_t smem_bytes() {
        return sizeof(T) * ((size_t)WENO_DEPTH * STAGE + WENO_ROWS * NH * RWX + NF * WENO_THREADS +
                            2 * RING * WENO_THREADS);
    }
};

template <class T, int R, int EOS>
__global__ void __launch_bounds__(WENO_THREADS, (R == 4 && sizeof(T) == 8) ? 2 : WENO5_MINB)
weno_xz_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* Un, T* Uout, Ctl* ctl, int zc) {
    using S = WenoXZShape<T, R>;
    using Win = typename S::Win;
    constexpr int M = 2 * R, NV = S::NV, NS = S::NS, NH = S::NH, NHL = S::NHL, RWX = S::RWX, D = WENO_DEPTH;
    constexpr int TH = WENO_THREADS, RING = S::RING;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);
    const int lane = threadIdx.x, wy = threadIdx.y, tid = wy * 32 + lane;
    const int i0 = (int)blockIdx.x * 31 - 1, i = i0 + lane;
    const int j = (int)blockIdx.y * WENO_ROWS + wy;
    if (j >= G.n[1]) return;   // whole warp
    T* row = sm + D * S::STAGE + wy * NH * RWX;            // [NH][RWX], this warp's
    T* park = sm + D * S::STAGE + WENO_ROWS * NH * RWX + tid; // [NF][TH]: this thread's last z-flux
    T* ring = sm + D * S::STAGE + WENO_ROWS * NH * RWX + NF * TH + tid;   // [RING][2][TH]: this thread's (v_x, a_x)
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
    const int dirs_zx[2] = {2, 0}, dirs_x[1] = {0};
    // the helper lane and the idle lanes of a ragged last tile march through x-ghost columns, whose z-ghost cells
    // are edge ghosts nobody fills (zeros): the flag their con2prim raises there is discarded
    int flag = 0;
    auto counts = [&](int plane) { return own || (plane >= 0 && plane < G.n[2]); };

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

    // a cell entering the z window: its conserved values -> (u, v_z, p, a_z) for the window and (v_x, a_x) into the
    // ring slot of its plane
    auto enter = [&](const T u[NF], T cell[NV], int slot, int& fl) {
        T v[2], a[2], p;
        cell_prims<T, 2, EOS>(u, A.eos, dirs_zx, v, a, p, fl);
#pragma unroll
        for (int c = 0; c < NF; ++c) cell[c] = u[c];
        cell[NF] = v[0];
        cell[NF + 1] = p;
        cell[NF + 2] = a[0];
        ring[(slot * 2 + 0) * TH] = v[1];
        ring[(slot * 2 + 1) * TH] = a[1];
    };

    Win zw;
    T nxt[NV];
#pragma unroll
    for (int m = 0; m < M; ++m) {   // cells k0-R .. k0+R-1; planes k0 .. k0+R-1 take ring slots 0 .. R-1
        T u[NF];
#pragma unroll
        for (int c = 0; c < NF; ++c) u[c] = __ldg(Us + c * G.fs + p0 + (long long)(m - R) * G.sxy);
        int fl = 0;
        enter(u, nxt, m >= R ? m - R : RING - 1, fl);   // (planes below k0: the slot is overwritten before it is read)
        if (counts(k0 - R + m)) flag |= fl;
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

    int rs = 0, ws = R;   // ring slots of plane k (read) and of plane k+R (written)
    for (int k = k0; k < k1; ++k) {
        cp_async_wait<D - 1>();   // plane k's stage has landed
        const T* st = sm + ((k - k0) % D) * S::STAGE;
        const T* src = st + tid;
        {
            T u[NF];
#pragma unroll
            for (int c = 0; c < NF; ++c) u[c] = src[c * TH];
            int fl = 0;
            enter(u, nxt, ws, fl);      // cell k+R: a z-ghost (possibly an unfilled edge ghost) in the last planes
            if (counts(k + R)) flag |= fl;
        }
        zw.shift();
        zw.put(M - 1, nxt);
        __syncwarp();             // every lane is done with the row of plane k-1
#pragma unroll
        for (int c = 0; c < NF; ++c) row[c * RWX + lane + R - 1] = zw.uu[c][R - 1];
        row[(NF + 0) * RWX + lane + R - 1] = ring[(rs * 2 + 0) * TH];
        row[(NF + 1) * RWX + lane + R - 1] = zw.ww[1][R - 1];
        row[(NF + 2) * RWX + lane + R - 1] = ring[(rs * 2 + 1) * TH];
        if (lane < NHL) {   // the halo cells: conserved values from their slots, (v_x, p, a_x) made here
            const T* hs = st + NS * TH + (wy * NHL + lane) * NF;
            T u[NF], v[1], a[1], p;
#pragma unroll
            for (int c = 0; c < NF; ++c) u[c] = hs[c];
            cell_prims<T, 1, EOS>(u, A.eos, dirs_x, v, a, p, flag);
#pragma unroll
            for (int c = 0; c < NF; ++c) row[c * RWX + hq] = u[c];
            row[(NF + 0) * RWX + hq] = v[0];
            row[(NF + 1) * RWX + hq] = p;
            row[(NF + 2) * RWX + hq] = a[0];
        }
        __syncwarp();
        rs = rs + 1 == RING ? 0 : rs + 1;
        ws = ws + 1 == RING ? 0 : ws + 1;
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
                    if (use_un) v = tfma(ca, src[(NF + c) * TH], cb * v);   // u^n: read late, it is only needed here
                    Uout[c * G.fs + q] = v;
                }
            }
        }
        issue(k + D);             // refill the slot just consumed
    }
    if (flag) ctl->flag = 1;
}

// ---------------------------------------------------------------------------------------------------------
template <class T, int R>
constexpr size_t weno_y_smem_bytes() {
    return sizeof(T) * ((size_t)WENO_DEPTH * (NF + NF) + NF) * WENO_THREADS;
}

template <class T, int R, bool EPI, int EOS>
__global__ void __launch_bounds__(WENO_THREADS, (R == 4 && sizeof(T) == 8) ? 2 : WENO5_MINB)
weno_y_kernel(Geom G, StageArgs A, const T* __restrict__ Us, T* Uout, Ctl* ctl, int yc) {
    using Win = WenoWindow<T, R, 1>;
    constexpr int M = 2 * R, NV = Win::NV, NVO = NF + NF, D = WENO_DEPTH, TH = WENO_THREADS;
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
    const int dirs_y[1] = {1};
    int flag = 0;
    auto issue = [&](int j) {   // conserved values of window cell j+R and the old output of cell j
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

    auto enter = [&](const T u[NF], T cell[NV]) {
        T v[1], a[1], p;
        cell_prims<T, 1, EOS>(u, A.eos, dirs_y, v, a, p, flag);
#pragma unroll
        for (int c = 0; c < NF; ++c) cell[c] = u[c];
        cell[NF] = v[0];
        cell[NF + 1] = p;
        cell[NF + 2] = a[0];
    };

    Win yw;
    T nxt[NV];
#pragma unroll
    for (int m = 0; m < M; ++m) {
        T u[NF];
#pragma unroll
        for (int c = 0; c < NF; ++c) u[c] = __ldg(Us + c * G.fs + p0 + (long long)(m - R) * ms);
        enter(u, nxt);
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
    double amax = 0.0;
    for (int j = j0; j < j1; ++j) {
        T f[NF], o[NF];
        cp_async_wait<D - 1>();   // the oldest stage (cell j) has landed
        const T* src = sm + ((j - j0) % D) * NVO * TH + tid;
        {
            T u[NF];
#pragma unroll
            for (int c = 0; c < NF; ++c) u[c] = src[c * TH];
            enter(u, nxt);
        }
        yw.shift();
        yw.put(M - 1, nxt);
        llf_weno_iface2<T, R, 1>(yw, eps, f);
        const long long q = p0 + (long long)(j - j0) * ms;
#pragma unroll
        for (int c = 0; c < NF; ++c) {
            o[c] = tfma(coef, park[c * TH] - f[c], src[(NF + c) * TH]);   // old output: read late
            Uout[c * G.fs + q] = o[c];
            park[c * TH] = f[c];
        }
        issue(j + D);             // refill the slot just consumed
        if (EPI) {   // stage 3 of a CFL step: a4 of the finished cell (all three axes are active here)
            amax = fmax(amax, (double)max_speed_of_cell_t<T, EOS>(o, A.eos, true, true, true, flag));   // (fmax drops a NaN)
        }
    }
    if (EPI) warp_max_to(amax, &ctl->maxspeed_next_bits, wmask);
    if (flag) ctl->flag = 1;
}

template <class T, int R>
int configure_weno(char* err, size_t errlen) {
    const int sxz = (int)WenoXZShape<T, R>::smem_bytes(), sy = (int)weno_y_smem_bytes<T, R>();
    const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
    cudaError_t e = cudaFuncSetAttribute(weno_xz_kernel<T, R, 0>, attr, sxz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(weno_xz_kernel<T, R, 1>, attr, sxz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(weno_y_kernel<T, R, false, 0>, attr, sy);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(weno_y_kernel<T, R, true, 0>, attr, sy);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(weno_y_kernel<T, R, false, 1>, attr, sy);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(weno_y_kernel<T, R, true, 1>, attr, sy);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(weno_xz_kernel<T, R, 2>, attr, sxz);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(weno_y_kernel<T, R, false, 2>, attr, sy);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(weno_y_kernel<T, R, true, 2>, attr, sy);
    if (e != cudaSuccess) {
        snprintf(err, errlen, "cudaFuncSetAttribute (weno): %s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

// stage = x/z kernel over the planes [A.kbeg, A.kend) (writes Uout) + y sweep (adds L_y; stage 3 of a CFL step: the
// max signal speed of the new state).  parts: bit 0 the x/z kernel, bit 1 the y sweep.
template <class T, int R, int EOS>
void launch_weno_eos(const Geom& G, const StageArgs& A, const T* Us, const T* Un, T* Uout, Ctl* ctl, int zc, int yc,
                     cudaStream_t st, int parts, int* launches) {
    const dim3 b(32, WENO_ROWS, 1);
    if ((parts & 1) && A.kend > A.kbeg) {
        const dim3 g((G.n[0] + 30) / 31, (G.n[1] + WENO_ROWS - 1) / WENO_ROWS, (A.kend - A.kbeg + zc - 1) / zc);
        weno_xz_kernel<T, R, EOS><<<g, b, WenoXZShape<T, R>::smem_bytes(), st>>>(G, A, Us, Un, Uout, ctl, zc);
        ++*launches;
    }
    if (parts & 2) {
        const dim3 gy((G.n[0] + 31) / 32, (G.n[2] + WENO_ROWS - 1) / WENO_ROWS, (G.n[1] + yc - 1) / yc);
        if (A.epi_max && A.mode != 1)
            weno_y_kernel<T, R, true, EOS><<<gy, b, weno_y_smem_bytes<T, R>(), st>>>(G, A, Us, Uout, ctl, yc);
        else
            weno_y_kernel<T, R, false, EOS><<<gy, b, weno_y_smem_bytes<T, R>(), st>>>(G, A, Us, Uout, ctl, yc);
        ++*launches;
    }
}

template <class T, int R>
int launch_weno(const Geom& G, const StageArgs& A, const T* Us, const T* Un, T* Uout, Ctl* ctl, int zc, int yc,
                cudaStream_t st, int parts, int* launches, char* err, size_t errlen) {
    *launches = 0;
    if (A.eos.kind == 1) launch_weno_eos<T, R, 1>(G, A, Us, Un, Uout, ctl, zc, yc, st, parts, launches);
    else if (A.eos.kind == 2) launch_weno_eos<T, R, 2>(G, A, Us, Un, Uout, ctl, zc, yc, st, parts, launches);
    else launch_weno_eos<T, R, 0>(G, A, Us, Un, Uout, ctl, zc, yc, st, parts, launches);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(err, errlen, "%s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

}  // namespace hydro
