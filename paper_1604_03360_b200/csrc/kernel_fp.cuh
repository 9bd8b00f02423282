// kernel_fp.cuh -- FIELD-PARALLEL stage kernels of the WENO schemes: L(u) of Eq. (2)
// fused with the SSP-RK3 combination (a9) and with con2prim + signal speeds + the CFL
// max of the finished cells (a2-a4).  DESIGN.md section 7.
//
// Component-wise Lax-Friedrichs splitting (reading Q3) couples the five fields of an interface only through
// per-CELL quantities: the velocity v_d, the pressure and the signal speed a_d, all made once per stage by the
// previous stage's epilogue.  So a THREAD OWNS ONE FIELD of one grid column: a block is 32 x-positions x 5 fields
// (one warp per field).  Against one thread carrying all five fields this cuts the live stencil from 48 to
// 24 values, which lets 20 warps (instead of 12) share an SM: the fp64 pipe, which a dependent instruction can
// only re-enter every 8 cycles, is kept busy by more independent warps.
//
// The split fluxes are f+- = F +- alpha u with F the field's physical flux (a5) and alpha the interface's own
// maximum of a_d (a6), so their first differences -- all the reconstruction needs -- are ONE fused multiply-add
// from the differences of F and of u, which do not depend on the interface and are carried in the marching window
// (llf_weno_field2 in iface.cuh): no split flux is ever formed.
//
//   fp_y_kernel<T, R>         marches along y; thread = (x, z, field).  Writes P = u_s + dt L_y (or L_y, mode 1).
//   fp_xz_kernel<T, R, EPI>   marches along z with the z-stencil in the window; the x-stencil of plane k comes
//                             from a per-WARP shared-memory row that every lane fills with its own cell (F_x, u, a_x)
//                             and 2r-1 halo lanes extend; the lower x-face comes from lane-1 by shuffle.  Finishes
//                             the stage: out = ca u^n + cb (P + dt (L_x + L_z)).  EPI: the five field-warps of a
//                             block exchange their finished values through shared memory once per five planes (one
//                             block barrier), and each warp then runs con2prim + signal speeds (a2-a3) for ONE of
//                             the five planes: the next stage's primitives W' and, in stage 3, the CFL max (a4).
// Every global read of the loops is a cp.async into the thread's own slots FP_DEPTH cells ahead (pipeline.cuh).
#pragma once
#include <cstdio>

#include "grid.cuh"
#include "iface.cuh"
#include "kernel_generic.cuh"
#include "kernels_aux.cuh"
#include "pipeline.cuh"

namespace hydro {

constexpr int FP_THREADS = 32 * NF;   // one warp per field
constexpr int FP_DEPTH = 3;           // cells in flight per thread
constexpr int FP_YC = 128, FP_ZC = 128;   // default cells per chunk of the y / z march ("sweep_zc" / "tile_zc")

// physical flux of one field along the marched axis from the cell's values (a5): kind 0 energy (F = M_d, loaded
// as such), 1 the momentum along the axis (F = M_d v_d + p), 2 transverse momenta and charge (F = u v_d)
template <class T>
__device__ __forceinline__ T field_flux(int kind, T u, T vf, T p) {
    return kind == 0 ? vf : (kind == 1 ? tfma(u, vf, p) : u * vf);
}

// marching window of ONE field along one axis: for the 2r stencil cells of the current interface the differences
// of F and u of the 2r-1 neighbouring pairs, F and u of cells r-1 .. 2r-1, and a_d of all of them
template <class T, int R>
struct FieldWindow {
    static constexpr int M = 2 * R, P = 2 * R - 1;
    T F[R + 1], u[R + 1], dF[P], du[P], a[M];
    __device__ __forceinline__ void first(T Fn, T un, T an) {
#pragma unroll
        for (int j = 0; j < P; ++j) dF[j] = du[j] = (T)0;
#pragma unroll
        for (int j = 0; j <= R; ++j) F[j] = u[j] = (T)0;
#pragma unroll
        for (int j = 0; j < M; ++j) a[j] = (T)0;
        F[R] = Fn;
        u[R] = un;
        a[M - 1] = an;
    }
    __device__ __forceinline__ void push(T Fn, T un, T an) {
#pragma unroll
        for (int j = 0; j + 1 < P; ++j) {
            dF[j] = dF[j + 1];
            du[j] = du[j + 1];
        }
        dF[P - 1] = Fn - F[R];
        du[P - 1] = un - u[R];
#pragma unroll
        for (int j = 0; j < R; ++j) {
            F[j] = F[j + 1];
            u[j] = u[j + 1];
        }
        F[R] = Fn;
        u[R] = un;
#pragma unroll
        for (int j = 0; j + 1 < M; ++j) a[j] = a[j + 1];
        a[M - 1] = an;
    }
    // twice the interface flux between stencil cells r-1 and r (a6-a7)
    __device__ __forceinline__ T flux2(T eps) const {
        T al = a[0];
#pragma unroll
        for (int k = 1; k < M; ++k) al = max_nonneg(al, a[k]);
        return llf_weno_field2<T, R>(dF, du, F[0] + F[1], al, eps);
    }
};

// ---------------------------------------------------------------------------------------------------------
template <class T>
constexpr size_t fp_y_smem_bytes() { return sizeof(T) * (size_t)FP_DEPTH * 4 * FP_THREADS; }

template <class T, int R>
__global__ void __launch_bounds__(FP_THREADS, (R == 4 && sizeof(T) == 8) ? 3 : 4)
fp_y_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* __restrict__ W, T* __restrict__ Pout, Ctl* ctl,
            int yc) {
    constexpr int M = 2 * R, D = FP_DEPTH, NS = 4, TH = FP_THREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);   // [D][NS][TH]
    const int lane = threadIdx.x, c = threadIdx.y, tid = c * 32 + lane;
    const int i = blockIdx.x * 32 + lane, kz = blockIdx.y;
    const bool active = i < G.n[0];
    const int j0 = (int)blockIdx.z * yc;
    const int j1 = min(j0 + yc, G.n[1]);
    const long long ms = G.sx;
    const long long p0 = G.pidx(min(i, G.n[0] - 1), j0, kz);
    const int kind = c == 0 ? 0 : (c == 2 ? 1 : 2);
    const T* pu = Us + c * G.fs;
    const T* pvf = c == 0 ? Us + 2 * G.fs : W + (W_V + 1) * G.fs;   // energy: F = M_y itself
    const T* pa = W + (W_AX + 1) * G.fs;
    const T* pp = W + W_P * G.fs;
    auto issue = [&](int j) {   // cell j + R of the march
        if (j < j1) {
            T* dst = sm + ((j - j0) % D) * NS * TH + tid;
            const long long q = p0 + (long long)(j - j0 + R) * ms;
            cp_async<sizeof(T)>(dst, pu + q);
            cp_async<sizeof(T)>(dst + TH, pvf + q);
            cp_async<sizeof(T)>(dst + 2 * TH, pa + q);
            if (kind == 1) cp_async<sizeof(T)>(dst + 3 * TH, pp + q);
        }
        cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d < D; ++d) issue(j0 + d);

    FieldWindow<T, R> win;
#pragma unroll
    for (int m = 0; m < M; ++m) {   // cells j0-R .. j0+R-1
        const long long q = p0 + (long long)(m - R) * ms;
        const T un = __ldg(pu + q), vf = __ldg(pvf + q), an = __ldg(pa + q);
        const T pn = kind == 1 ? __ldg(pp + q) : (T)0;
        const T Fn = field_flux(kind, un, vf, pn);
        if (m == 0) win.first(Fn, un, an);
        else win.push(Fn, un, an);
    }
    const T eps = (T)A.eps;
    T f_lo = win.flux2(eps);   // face j0 - 1/2
    // the 1/2 of the Lax-Friedrichs split is folded into the step factor
    const T hdt = (T)(A.mode == 1 ? 0.5 * A.inv_dx : 0.5 * ctl->dt * A.inv_dx);
    for (int j = j0; j < j1; ++j) {
        cp_async_wait<D - 1>();   // cell j + R has landed
        const T* src = sm + ((j - j0) % D) * NS * TH + tid;
        const T un = src[0], vf = src[TH], an = src[2 * TH];
        const T pn = kind == 1 ? src[3 * TH] : (T)0;
        issue(j + D);             // refill the slot just consumed
        win.push(field_flux(kind, un, vf, pn), un, an);
        const T f_hi = win.flux2(eps);
        const T d = f_lo - f_hi;
        f_lo = f_hi;
        const T out = A.mode == 1 ? hdt * d : tfma(hdt, d, win.u[0]);
        if (active) Pout[c * G.fs + p0 + (long long)(j - j0) * ms] = out;
    }
}

// ---------------------------------------------------------------------------------------------------------
template <class T, int R>
struct FpXZShape {
    static constexpr int D = FP_DEPTH, TH = FP_THREADS;
    static constexpr int NS = 8;                  // slots per thread: u, vf_z, a_z of cell k+R; p; vf_x, a_x, P, u^n of plane k
    static constexpr int NHL = 2 * R - 1;         // halo lanes: R-1 cells below, R cells above the row
    static constexpr int NHV = 4;                 // per halo cell: u, vf_x, a_x, p
    static constexpr int RWX = 32 + 2 * R - 1;    // cells of a row with halo
    static constexpr int STAGE = NS * TH + NF * NHL * NHV;
    static constexpr int ROWS = NF * 3 * RWX;     // per warp: F_x, u, a_x
    static constexpr int EXCH = 2 * NF * NF * 32; // [2][plane of the batch][field][lane]
    static constexpr size_t smem_bytes(bool epi) {
        return sizeof(T) * ((size_t)D * STAGE + ROWS + (epi ? EXCH : 0));
    }
};

template <class T, int R, bool EPI>
__global__ void __launch_bounds__(FP_THREADS, (R == 4 && sizeof(T) == 8) ? 3 : 4)
fp_xz_kernel(Geom G, StageArgs A, const T* __restrict__ Us, const T* __restrict__ W, const T* Pin, const T* Un,
             T* Uout, T* __restrict__ Wnext, Ctl* ctl, int zc) {
    using S = FpXZShape<T, R>;
    constexpr int M = 2 * R, D = S::D, TH = S::TH, NHL = S::NHL, NHV = S::NHV, RWX = S::RWX;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sm = reinterpret_cast<T*>(smem_raw);
    const int lane = threadIdx.x, c = threadIdx.y, tid = c * 32 + lane;
    const int i0 = (int)blockIdx.x * 31 - 1, i = i0 + lane;
    const int jy = blockIdx.y;
    T* row = sm + D * S::STAGE + c * 3 * RWX;   // this warp's [3][RWX]
    T* exch = sm + D * S::STAGE + S::ROWS;
    const bool own = lane >= 1 && i < G.n[0];
    const bool need_x = i < G.n[0];             // i >= -1 always
    const int imax = G.n[0] - 1 + G.g[0];
    const int hcell = lane < R - 1 ? i0 - (R - 1) + lane : i0 + 32 + (lane - (R - 1));   // halo lanes' column
    const int hq = lane < R - 1 ? lane : 32 + lane;                                        // and its row position
    const int k0 = (int)blockIdx.z * zc;
    const int k1 = min(k0 + zc, G.n[2]);
    const long long p0 = G.pidx(min(i, imax), jy, k0);
    const long long ph = G.pidx(min(hcell, imax), jy, k0);
    const int kindz = c == 0 ? 0 : (c == 3 ? 1 : 2), kindx = c == 0 ? 0 : (c == 1 ? 1 : 2);
    const T* pu = Us + c * G.fs;
    const T* pvfz = c == 0 ? Us + 3 * G.fs : W + (W_V + 2) * G.fs;   // energy: F = M_d itself
    const T* pvfx = c == 0 ? Us + 1 * G.fs : W + (W_V + 0) * G.fs;
    const T* paz = W + (W_AX + 2) * G.fs;
    const T* pax = W + (W_AX + 0) * G.fs;
    const T* pp = W + W_P * G.fs;
    const bool use_un = A.mode != 1 && A.ca != 0.0;

    auto issue = [&](int k) {
        if (k < k1) {
            T* st = sm + ((k - k0) % D) * S::STAGE;
            T* dst = st + tid;
            const long long q = p0 + (long long)(k - k0) * G.sxy, qr = q + (long long)R * G.sxy;
            cp_async<sizeof(T)>(dst, pu + qr);
            cp_async<sizeof(T)>(dst + TH, pvfz + qr);
            cp_async<sizeof(T)>(dst + 2 * TH, paz + qr);
            if (kindz == 1) cp_async<sizeof(T)>(dst + 3 * TH, pp + qr);
            if (kindx == 1) cp_async<sizeof(T)>(dst + 3 * TH, pp + q);
            cp_async<sizeof(T)>(dst + 4 * TH, pvfx + q);
            cp_async<sizeof(T)>(dst + 5 * TH, pax + q);
            cp_async<sizeof(T)>(dst + 6 * TH, Pin + c * G.fs + q);
            if (use_un) cp_async<sizeof(T)>(dst + 7 * TH, Un + c * G.fs + q);
            if (lane < NHL) {
                T* hd = st + S::NS * TH + (c * NHL + lane) * NHV;
                const long long qh = ph + (long long)(k - k0) * G.sxy;
                cp_async<sizeof(T)>(hd, pu + qh);
                cp_async<sizeof(T)>(hd + 1, pvfx + qh);
                cp_async<sizeof(T)>(hd + 2, pax + qh);
                if (kindx == 1) cp_async<sizeof(T)>(hd + 3, pp + qh);
            }
        }
        cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d < D; ++d) issue(k0 + d);

    FieldWindow<T, R> win;
#pragma unroll
    for (int m = 0; m < M; ++m) {   // cells k0-R .. k0+R-1
        const long long q = p0 + (long long)(m - R) * G.sxy;
        const T un = __ldg(pu + q), vf = __ldg(pvfz + q), an = __ldg(paz + q);
        const T pn = kindz == 1 ? __ldg(pp + q) : (T)0;
        const T Fn = field_flux(kindz, un, vf, pn);
        if (m == 0) win.first(Fn, un, an);
        else win.push(Fn, un, an);
    }
    const T eps = (T)A.eps;
    T fz_lo = win.flux2(eps);   // face k0 - 1/2
    const T hdt = (T)(A.mode == 1 ? 0.5 * A.inv_dx : 0.5 * ctl->dt * A.inv_dx);
    const T ca = (T)A.ca, cb = (T)A.cb;
    int flag = 0, buf = 0;
    double amax = 0.0;

    for (int k = k0; k < k1; ++k) {
        cp_async_wait<D - 1>();   // plane k's stage has landed
        const T* st = sm + ((k - k0) % D) * S::STAGE;
        const T* src = st + tid;
        const T un = src[0], vfz = src[TH], azn = src[2 * TH];
        const T pv = (kindz == 1 || kindx == 1) ? src[3 * TH] : (T)0;
        const T vfx = src[4 * TH], axk = src[5 * TH], Pk = src[6 * TH];
        const T unk = use_un ? src[7 * TH] : (T)0;
        T hu = (T)0, hvf = (T)0, ha = (T)0, hp = (T)0;
        if (lane < NHL) {
            const T* hs = st + S::NS * TH + (c * NHL + lane) * NHV;
            hu = hs[0];
            hvf = hs[1];
            ha = hs[2];
            if (kindx == 1) hp = hs[3];
        }
        issue(k + D);             // refill the slot just consumed
        win.push(field_flux(kindz, un, vfz, kindz == 1 ? pv : (T)0), un, azn);
        const T uk = win.u[0];    // this column's cell of plane k
        __syncwarp();             // every lane is done with the row of plane k-1
        row[lane + R - 1] = field_flux(kindx, uk, vfx, kindx == 1 ? pv : (T)0);
        row[RWX + lane + R - 1] = uk;
        row[2 * RWX + lane + R - 1] = axk;
        if (lane < NHL) {
            row[hq] = field_flux(kindx, hu, hvf, hp);
            row[RWX + hq] = hu;
            row[2 * RWX + hq] = ha;
        }
        __syncwarp();
        const T fz_hi = win.flux2(eps);
        T L2 = fz_lo - fz_hi;
        fz_lo = fz_hi;
        T fx = (T)0;
        if (need_x) {
            T Fr[M], ur[M], dF[M - 1], du[M - 1];
            T al = row[2 * RWX + lane];
#pragma unroll
            for (int m = 0; m < M; ++m) {
                Fr[m] = row[lane + m];
                ur[m] = row[RWX + lane + m];
                if (m > 0) al = max_nonneg(al, row[2 * RWX + lane + m]);
            }
#pragma unroll
            for (int m = 0; m + 1 < M; ++m) {
                dF[m] = Fr[m + 1] - Fr[m];
                du[m] = ur[m + 1] - ur[m];
            }
            fx = llf_weno_field2<T, R>(dF, du, Fr[R - 1] + Fr[R], al, eps);
        }
        L2 += shfl_up1<T>(fx) - fx;
        T out = tfma(hdt, L2, Pk);
        if (use_un) out = tfma(ca, unk, cb * out);
        const long long q = p0 + (long long)(k - k0) * G.sxy;
        if (own) Uout[c * G.fs + q] = out;
        if (EPI) {
            const int slot = (k - k0) % NF;
            exch[((buf * NF + slot) * NF + c) * 32 + lane] = out;
            if (slot == NF - 1 || k == k1 - 1) {
                __syncthreads();   // the five field-warps have written this batch of planes
                if (c <= slot) {   // warp c takes plane c of the batch: a2-a3 of its finished cells
                    T u5[NF], w[NW];
                    int fl = 0;
#pragma unroll
                    for (int f = 0; f < NF; ++f) u5[f] = exch[((buf * NF + c) * NF + f) * 32 + lane];
                    prim_of_cell(u5, w, fl, A.eos);
                    if (own) {
                        const long long qe = p0 + (long long)(k - slot + c - k0) * G.sxy;
#pragma unroll
                        for (int a = 0; a < NW; ++a) Wnext[a * G.fs + qe] = w[a];
                        if (A.epi_max)
                            amax = fmax(amax, fmax((double)w[W_AX], fmax((double)w[W_AX + 1], (double)w[W_AX + 2])));
                        flag |= fl;
                    }
                }
                buf ^= 1;
            }
        }
    }
    if (EPI && A.epi_max) warp_max_to(amax, &ctl->maxspeed_next_bits);   // all three axes are active here
    if (flag) ctl->flag = 1;
}

template <class T, int R>
int configure_fp(char* err, size_t errlen) {
    cudaError_t e = cudaFuncSetAttribute(fp_y_kernel<T, R>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)fp_y_smem_bytes<T>());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(fp_xz_kernel<T, R, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)FpXZShape<T, R>::smem_bytes(false));
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(fp_xz_kernel<T, R, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)FpXZShape<T, R>::smem_bytes(true));
    if (e != cudaSuccess) {
        snprintf(err, errlen, "cudaFuncSetAttribute (fp): %s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

// stage = y sweep (P = u_s + dt L_y into Pbuf) + x/z kernel (finishes the stage into Uout; epilogue -> Wnext).
// Pbuf may be Uout itself unless Uout is also u^n (stage 3, which writes u^n in place).
template <class T, int R>
int launch_fp(const Geom& G, const StageArgs& A, const T* Us, const T* W, const T* Un, T* Uout, T* Pbuf, T* Wnext,
              Ctl* ctl, int zc, int yc, cudaStream_t st, int* launches, char* err, size_t errlen) {
    const dim3 b(32, NF, 1);
    const dim3 gy((G.n[0] + 31) / 32, G.n[2], (G.n[1] + yc - 1) / yc);
    fp_y_kernel<T, R><<<gy, b, fp_y_smem_bytes<T>(), st>>>(G, A, Us, W, Pbuf, ctl, yc);
    const dim3 g((G.n[0] + 30) / 31, G.n[1], (G.n[2] + zc - 1) / zc);
    if (Wnext != nullptr && A.mode != 1)
        fp_xz_kernel<T, R, true><<<g, b, FpXZShape<T, R>::smem_bytes(true), st>>>(G, A, Us, W, Pbuf, Un, Uout, Wnext, ctl, zc);
    else
        fp_xz_kernel<T, R, false><<<g, b, FpXZShape<T, R>::smem_bytes(false), st>>>(G, A, Us, W, Pbuf, Un, Uout, nullptr, ctl, zc);
    *launches = 2;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(err, errlen, "%s", cudaGetErrorString(e));
        return -1;
    }
    return 0;
}

}  // namespace hydro
