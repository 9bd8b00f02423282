// kernels_aux.cuh -- the small kernels around the stage kernel:
//   (d) halo_fill_kernel    a1: outflow / periodic / analytic Hubble ghost fill, face ghosts only
//   (a) prim_kernel         a2-a4: con2prim + three signal speeds per padded cell, fused with the
//                           warp-shuffle / block / atomic max reduction for the CFL time step
//       max_speed_kernel    a4 alone (interior cells, no stores): hydro_max_signal_speed, MUSTA CFL mode
//       pack / unpack       interior <-> padded copies for hydro_set_state / hydro_get_state
//       begin_step / end_step  device-resident dt and t
#pragma once
#include "device_math.cuh"
#include "grid.cuh"

namespace hydro {

// ------------------------------------------------------------------------------------------------
// step control
__global__ void begin_step_kernel(Ctl* ctl, double dt_fixed, double cfl, double dx) {
    // dt_fixed > 0: fixed step.  Otherwise dt = cfl * dx / max signal speed reduced by the stage-1
    // prim / max-speed kernel (reading Q10).
    if (dt_fixed > 0.0) {
        ctl->dt = dt_fixed;
    } else {
        const double s = __longlong_as_double((long long)ctl->maxspeed_bits);
        ctl->dt = cfl * dx / s;
    }
}
__global__ void end_step_kernel(Ctl* ctl) {
    ctl->t += ctl->dt;
    // the stage-3 epilogue of the z sweep (when it ran) left the max signal speed of the new state here
    ctl->maxspeed_bits = ctl->maxspeed_next_bits;
    ctl->maxspeed_next_bits = 0ull;
}
__global__ void reset_max_kernel(Ctl* ctl) { ctl->maxspeed_bits = 0ull; }

// W = (winv, p, a_x, a_y, a_z) of one cell from its conserved values (a2-a3).  EOS 0: p = e/3; EOS 1: p = p0,
// whose characteristic speeds are all v_d, so a_d = |v_d|.
template <class T, int EOS>
__device__ __forceinline__ void prim_of_cell_t(const T u[NF], T w[NW], int& flag, T p0) {
    T v2;
    if (EOS == 1) {
        con2prim_p0(u[0], u[1], u[2], u[3], p0, w[W_INV], w[W_P], v2, flag);
        w[W_AX + 0] = tabs(u[1] * w[W_INV]);
        w[W_AX + 1] = tabs(u[2] * w[W_INV]);
        w[W_AX + 2] = tabs(u[3] * w[W_INV]);
    } else {
        con2prim(u[0], u[1], u[2], u[3], w[W_INV], w[W_P], v2, flag);
        const T id = speed_inv_den(v2);
        w[W_AX + 0] = signal_speed(u[1] * w[W_INV], v2, id);
        w[W_AX + 1] = signal_speed(u[2] * w[W_INV], v2, id);
        w[W_AX + 2] = signal_speed(u[3] * w[W_INV], v2, id);
    }
}
struct EosArgs {
    int kind;     // 0: p = e/3, 1: p = p0
    double p0;
};
template <class T>
__device__ __forceinline__ void prim_of_cell(const T u[NF], T w[NW], int& flag, const EosArgs& eos) {
    if (eos.kind == 1) prim_of_cell_t<T, 1>(u, w, flag, (T)eos.p0);
    else prim_of_cell_t<T, 0>(u, w, flag, (T)0);
}

// ------------------------------------------------------------------------------------------------
// pack: interior [5][nz][ny][nx] -> padded;  unpack: the reverse.  One thread per interior cell.
template <class T>
__global__ void pack_kernel(Geom G, const T* __restrict__ in, T* __restrict__ pad) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= G.n[0] || j >= G.n[1]) return;
    const long long N = (long long)G.n[0] * G.n[1] * G.n[2];
    const long long q = ((long long)k * G.n[1] + j) * G.n[0] + i, p = G.pidx(i, j, k);
#pragma unroll
    for (int c = 0; c < NF; ++c) pad[c * G.fs + p] = in[c * N + q];
}
template <class T>
__global__ void unpack_kernel(Geom G, const T* __restrict__ pad, T* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= G.n[0] || j >= G.n[1]) return;
    const long long N = (long long)G.n[0] * G.n[1] * G.n[2];
    const long long q = ((long long)k * G.n[1] + j) * G.n[0] + i, p = G.pidx(i, j, k);
#pragma unroll
    for (int c = 0; c < NF; ++c) out[c * N + q] = pad[c * G.fs + p];
}

// ------------------------------------------------------------------------------------------------
// (d) halo fill, a1 (reading Q9).  One thread per face-ghost cell; the three axes are independent
// because only face ghosts exist.  Ghost cells of axis a are enumerated as (q1, l, side, q2) with q1
// the lower-numbered other axis, so that for the y and z faces consecutive threads run along x.
// bc: per axis 0 outflow (copy the nearest interior cell), 1 periodic (wrap), 2 analytic Hubble flow
// at time ctl->t + tfrac * ctl->dt (stage times t, t+dt, t+dt/2, O8).
template <class T>
__device__ void hubble_cons(const HubbleParams& H, const int bc[3], int i, int j, int k, double tt, T out[NF]) {
    const int ix[3] = {i, j, k};
    double r2 = 0, s = 0, v[3] = {0, 0, 0};
    int d = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (bc[a] != 2) continue;
        const double x = H.origin[a] + (ix[a] + 0.5) * H.dx;
        ++d;
        r2 += x * x;
        v[a] = x / tt;
        if (H.b[a] > 0) s += (x / tt) * (x / tt) / (H.b[a] * H.b[a]);
    }
    const double tau = sqrt(tt * tt - r2);
    const double e = H.e0 * pow(H.t0 / tau, 4.0 * d / 3.0);
    const double nn = H.n0 * pow(H.t0 / tau, (double)d) * exp(-0.5 * s);
    const double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    const double g2 = 1.0 / (1.0 - v2), p = e / 3.0, w = (e + p) * g2;
    out[0] = (T)(w - p);
    out[1] = (T)(w * v[0]);
    out[2] = (T)(w * v[1]);
    out[3] = (T)(w * v[2]);
    out[4] = (T)(nn * sqrt(g2));
}

struct HaloArgs {
    EosArgs eos;
    int bc[3];
    long long count[3];  // ghost cells per axis
    HubbleParams H;
};

template <class T>
__global__ void halo_fill_kernel(Geom G, HaloArgs A, Ctl* ctl, double tfrac, double t_abs,
                                 int use_abs, T* __restrict__ pad, T* __restrict__ Wghost) {
    long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int a = 0;
    for (; a < 3; ++a) {
        if (id < A.count[a]) break;
        id -= A.count[a];
    }
    if (a == 3) return;
    const int a1 = a == 0 ? 1 : 0, a2 = a == 2 ? 1 : 2;  // the other two axes, lower first
    const int g = G.g[a];
    int ix[3], src[3];
    // id = ((q2 * 2 + side) * g + (l-1)) * n[a1] + q1   for y/z faces (q1 = x fastest)
    // for x faces (a = 0): id = ((q2 * n[a1] + q1) * 2 + side) * g + (l-1)
    int l, side, q1, q2;
    if (a == 0) {
        l = (int)(id % g) + 1; id /= g;
        side = (int)(id % 2); id /= 2;
        q1 = (int)(id % G.n[a1]); q2 = (int)(id / G.n[a1]);
    } else {
        q1 = (int)(id % G.n[a1]); id /= G.n[a1];
        l = (int)(id % g) + 1; id /= g;
        side = (int)(id % 2); q2 = (int)(id / 2);
    }
    ix[a1] = src[a1] = q1;
    ix[a2] = src[a2] = q2;
    ix[a] = side == 0 ? -l : G.n[a] - 1 + l;
    T val[NF];
    if (A.bc[a] == 3) {
        // external ghosts (slab decomposition): the caller put them there (hydro_put_zhalo); only their
        // primitives may have to be made below
        if (Wghost == nullptr) return;
        const long long pg = G.pidx(ix[0], ix[1], ix[2]);
#pragma unroll
        for (int c = 0; c < NF; ++c) val[c] = pad[c * G.fs + pg];
    } else if (A.bc[a] == 2) {
        const double tt = use_abs ? t_abs : ctl->t + tfrac * ctl->dt;
        hubble_cons<T>(A.H, A.bc, ix[0], ix[1], ix[2], tt, val);
    } else {
        if (A.bc[a] == 1) src[a] = side == 0 ? G.n[a] - l : l - 1;
        else src[a] = side == 0 ? 0 : G.n[a] - 1;
        const long long ps = G.pidx(src[0], src[1], src[2]);
#pragma unroll
        for (int c = 0; c < NF; ++c) val[c] = pad[c * G.fs + ps];
    }
    const long long p = G.pidx(ix[0], ix[1], ix[2]);
    if (A.bc[a] != 3) {
#pragma unroll
        for (int c = 0; c < NF; ++c) pad[c * G.fs + p] = val[c];
    }
    // when the interior primitives came from the previous stage's z-sweep epilogue, the ghost cells' are made here
    if (Wghost != nullptr) {
        T w[NW];
        int flag = 0;
        prim_of_cell(val, w, flag, A.eos);
#pragma unroll
        for (int a = 0; a < NW; ++a) Wghost[a * G.fs + p] = w[a];
        if (flag) ctl->flag = 1;
    }
}

// ------------------------------------------------------------------------------------------------
// block-wide max of a non-negative value, result pushed to ctl->maxspeed_bits by one atomic per block
__device__ __forceinline__ void block_max_to_ctl(double m, Ctl* ctl) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    __shared__ double smax[32];
    const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
    const int nw = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
    if ((tid & 31) == 0) smax[tid >> 5] = m;
    __syncthreads();
    if (tid < 32) {
        m = tid < nw ? smax[tid] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (tid == 0 && m > 0.0) atomicMax(&ctl->maxspeed_bits, (unsigned long long)__double_as_longlong(m));
    }
}

// (a) con2prim + signal speeds over the padded array (face ghosts included, edge/corner ghosts
// skipped), a2-a3; the max over INTERIOR cells and ACTIVE axes (a4) is reduced when do_max != 0.
// Writes W = (winv, p, a_x, a_y, a_z).
template <class T>
__global__ void __launch_bounds__(256) prim_kernel(Geom G, const T* __restrict__ U, T* __restrict__ W,
                                                   Ctl* ctl, int do_max, EosArgs eos) {
    const int pi = blockIdx.x * blockDim.x + threadIdx.x;
    const int pj = blockIdx.y * blockDim.y + threadIdx.y;
    const int pk = blockIdx.z;
    double m = 0.0;
    int flag = 0;
    if (pi < G.np[0] && pj < G.np[1]) {
        const int i = pi - G.g[0], j = pj - G.g[1], k = pk - G.g[2];
        const int out = (i < 0 || i >= G.n[0]) + (j < 0 || j >= G.n[1]) + (k < 0 || k >= G.n[2]);
        if (out <= 1) {
            const long long p = (long long)pk * G.sxy + (long long)pj * G.sx + pi;
            const T u[NF] = {U[p], U[G.fs + p], U[2 * G.fs + p], U[3 * G.fs + p], (T)0};
            T w[NW];
            prim_of_cell(u, w, flag, eos);
            const T ax = w[W_AX], ay = w[W_AX + 1], az = w[W_AX + 2];
#pragma unroll
            for (int a = 0; a < NW; ++a) W[a * G.fs + p] = w[a];
            if (do_max && out == 0) {
                if (G.g[0]) m = fmax(m, (double)ax);
                if (G.g[1]) m = fmax(m, (double)ay);
                if (G.g[2]) m = fmax(m, (double)az);
            }
        }
    }
    if (flag) ctl->flag = 1;
    if (do_max) block_max_to_ctl(m, ctl);
}

// a4 alone: interior cells only, nothing stored.
template <class T>
__global__ void __launch_bounds__(256) max_speed_kernel(Geom G, const T* __restrict__ U, Ctl* ctl, EosArgs eos) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    double m = 0.0;
    int flag = 0;
    if (i < G.n[0] && j < G.n[1]) {
        const long long p = G.pidx(i, j, k);
        const T u[NF] = {U[p], U[G.fs + p], U[2 * G.fs + p], U[3 * G.fs + p], (T)0};
        T w[NW];
        prim_of_cell(u, w, flag, eos);
        if (G.g[0]) m = fmax(m, (double)w[W_AX]);
        if (G.g[1]) m = fmax(m, (double)w[W_AX + 1]);
        if (G.g[2]) m = fmax(m, (double)w[W_AX + 2]);
    }
    if (flag) ctl->flag = 1;
    block_max_to_ctl(m, ctl);
}

}  // namespace hydro
