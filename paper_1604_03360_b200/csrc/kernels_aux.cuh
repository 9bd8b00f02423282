// kernels_aux.cuh -- the small kernels around the stage kernel:
//   (d) halo_fill_kernel    a1: outflow / periodic / analytic Hubble ghost fill, face ghosts only
//   (a) prim_kernel         a2-a4: con2prim + three signal speeds per padded cell, fused with the
//                           warp-shuffle / block / atomic max reduction for the CFL time step (the GENERIC
//                           kernel's primitives; the marching kernels make theirs on the fly)
//       max_speed_kernel    a4 alone (interior cells, no stores): hydro_max_signal_speed
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
// the same with the max signal speed taken from a caller's device scalar (a double): the slab decomposition passes
// the value it has max-reduced over all slabs (reading Q10 on the global grid)
__global__ void begin_step_ext_kernel(Ctl* ctl, double cfl, double dx, const double* __restrict__ maxspeed) {
    ctl->dt = cfl * dx / *maxspeed;
}
__global__ void end_step_kernel(Ctl* ctl) {
    ctl->t += ctl->dt;
    // the stage-3 epilogue of the z sweep (when it ran) left the max signal speed of the new state here
    ctl->maxspeed_bits = ctl->maxspeed_next_bits;
    ctl->maxspeed_next_bits = 0ull;
}
__global__ void reset_max_kernel(Ctl* ctl) { ctl->maxspeed_bits = 0ull; }

// W = (v_x, v_y, v_z, p, a_x, a_y, a_z) of one cell from its conserved values (a2-a3).  EOS 0: p = e/3; EOS 1:
// p = p0, whose characteristic speeds are all v_d, so a_d = |v_d|; EOS 2: the tabulated closure.
template <class T, int EOS>
__device__ __forceinline__ void prim_of_cell_t(const T u[NF], T w[NW], int& flag, const EosArgs& eos) {
    T v2, winv, cs2;
    if (EOS == 1) con2prim_p0(u[0], u[1], u[2], u[3], (T)eos.p0, winv, w[W_P], v2, flag);
    else if (EOS == 2) con2prim_tab(u[0], u[1], u[2], u[3], eos, winv, w[W_P], v2, cs2, flag);
    else con2prim(u[0], u[1], u[2], u[3], winv, w[W_P], v2, flag);
#pragma unroll
    for (int d = 0; d < 3; ++d) w[W_V + d] = u[1 + d] * winv;
    if (EOS == 1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) w[W_AX + d] = tabs(w[W_V + d]);
    } else if (EOS == 2) {
#pragma unroll
        for (int d = 0; d < 3; ++d) w[W_AX + d] = signal_speed_cs(w[W_V + d], v2, cs2);
    } else {
        const T id = speed_inv_den(v2);
#pragma unroll
        for (int d = 0; d < 3; ++d) w[W_AX + d] = signal_speed(w[W_V + d], v2, id);
    }
}
// a4 of one cell: the largest a_d over the axes flagged active.  For a given state a_d increases with |v_d|
// (d a_d / d|v_d| = (1 - cs2)(1 - cs (1 - v^2)|v_d| / sqrt(disc)) > 0, because cs2 (1 - v^2) v_d^2 < disc reduces to
// (1 - v_d^2)(1 - v^2 cs2) > 0), so it is the speed of the axis with the largest |M_d|: one speed, not three.
template <class T, int EOS>
__device__ __forceinline__ T max_speed_of_cell_t(const T u[NF], const EosArgs& eos, bool ax, bool ay, bool az,
                                                 int& flag) {
    T v2, winv, p, cs2;
    if (EOS == 1) con2prim_p0(u[0], u[1], u[2], u[3], (T)eos.p0, winv, p, v2, flag);
    else if (EOS == 2) con2prim_tab(u[0], u[1], u[2], u[3], eos, winv, p, v2, cs2, flag);
    else con2prim(u[0], u[1], u[2], u[3], winv, p, v2, flag);
    T m = (T)0;
    if (ax) m = max_nonneg(m, tabs(u[1]));
    if (ay) m = max_nonneg(m, tabs(u[2]));
    if (az) m = max_nonneg(m, tabs(u[3]));
    if (!(ax || ay || az)) return (T)0;   // no active axis: nothing enters the maximum (a4)
    const T vd = m * winv;
    if (EOS == 1) return vd;
    if (EOS == 2) return signal_speed_cs(vd, v2, cs2);
    return signal_speed(vd, v2, speed_inv_den(v2));
}
template <class T>
__device__ __forceinline__ T max_speed_of_cell(const T u[NF], const EosArgs& eos, bool ax, bool ay, bool az, int& flag) {
    if (eos.kind == 1) return max_speed_of_cell_t<T, 1>(u, eos, ax, ay, az, flag);
    if (eos.kind == 2) return max_speed_of_cell_t<T, 2>(u, eos, ax, ay, az, flag);
    return max_speed_of_cell_t<T, 0>(u, eos, ax, ay, az, flag);
}

template <class T>
__device__ __forceinline__ void prim_of_cell(const T u[NF], T w[NW], int& flag, const EosArgs& eos) {
    if (eos.kind == 1) prim_of_cell_t<T, 1>(u, w, flag, eos);
    else if (eos.kind == 2) prim_of_cell_t<T, 2>(u, w, flag, eos);
    else prim_of_cell_t<T, 0>(u, w, flag, eos);
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
// (d) halo fill, a1 (reading Q9).  One thread per face-ghost cell; the three axes are independent because only face
// ghosts exist.  A ghost cell of axis a is (m, q1, q2): m = 0 .. 2g-1 numbers the ghost coordinates
// -g .. -1, n .. n+g-1 in increasing order, q1 / q2 are the interior coordinates along the lower / higher of the
// other two axes; for the y and z faces consecutive threads run along x.
// bc per axis: 0 outflow (the coordinate is clamped into the interior: every ghost layer repeats the boundary cell),
// 1 periodic (the coordinate is taken modulo n), 2 analytic Hubble flow at time ctl->t + tfrac * ctl->dt (stage
// times t, t+dt, t+dt/2, O8), 3 external (z only: the caller wrote the planes, hydro_put_zhalo).

// Closed-form d-dimensional Hubble flow (readings Q13, Q14) in conserved variables, written from the invariants of
// the flow: with r^2 = sum of x_a^2 over the Hubble axes, tau^2 = t^2 - r^2 and gamma^2 = t^2 / tau^2,
//   e = e0 q^(2d/3),  n = n0 q^(d/2) exp(-sigma/2),  q = t0^2 / tau^2,  sigma = sum (x_a / (b_a t))^2  (b_a > 0),
//   E = e (3 t^2 + r^2) / (3 tau^2),  M_a = 4 e t x_a / (3 tau^2),  R = n t / tau.
template <class T>
__device__ void hubble_state(const HubbleParams& H, const int bc[3], const int cell[3], double t, T out[NF]) {
    double x[3], r2 = 0.0, sigma = 0.0;
    int d = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const bool on = bc[a] == 2;
        x[a] = on ? fma((double)cell[a] + 0.5, H.dx, H.origin[a]) : 0.0;
        d += on ? 1 : 0;
        r2 = fma(x[a], x[a], r2);
        if (on && H.b[a] > 0.0) {
            const double z = x[a] / (H.b[a] * t);
            sigma = fma(z, z, sigma);
        }
    }
    const double tau2 = t * t - r2, itau2 = 1.0 / tau2;
    const double q = H.t0 * H.t0 * itau2;
    const double e = H.e0 * pow(q, (2.0 / 3.0) * d);
    const double n = H.n0 * pow(q, 0.5 * d) * exp(-0.5 * sigma);
    const double k = (4.0 / 3.0) * e * t * itau2;
    out[0] = (T)(e * (3.0 * t * t + r2) * itau2 * (1.0 / 3.0));
    out[1] = (T)(k * x[0]);
    out[2] = (T)(k * x[1]);
    out[3] = (T)(k * x[2]);
    out[4] = (T)(n * t * sqrt(itau2));
}

struct HaloArgs {
    EosArgs eos;
    int bc[3];
    long long count[3];  // ghost cells per axis
    HubbleParams H;
};

template <class T>
__global__ void halo_fill_kernel(Geom G, HaloArgs A, Ctl* ctl, double tfrac, double t_abs,
                                 int use_abs, T* __restrict__ pad) {
    long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int a = 0;
    for (; a < 3; ++a) {
        if (id < A.count[a]) break;
        id -= A.count[a];
    }
    if (a == 3) return;
    const int a1 = a == 0 ? 1 : 0, a2 = a == 2 ? 1 : 2;  // the other two axes, lower first
    const int g = G.g[a], n = G.n[a];
    int m, q1, q2;
    if (a == 0) {   // x faces: m fastest
        m = (int)(id % (2 * g)); id /= 2 * g;
        q1 = (int)(id % G.n[a1]); q2 = (int)(id / G.n[a1]);
    } else {        // y and z faces: x fastest
        q1 = (int)(id % G.n[a1]); id /= G.n[a1];
        m = (int)(id % (2 * g)); q2 = (int)(id / (2 * g));
    }
    int cell[3];
    cell[a1] = q1;
    cell[a2] = q2;
    cell[a] = m < g ? m - g : n + (m - g);
    const long long p = G.pidx(cell[0], cell[1], cell[2]);
    if (A.bc[a] == 3) return;   // external ghosts (slab decomposition): the caller's business (hydro_put_zhalo)
    T val[NF];
    if (A.bc[a] == 2) {
        const double tt = use_abs ? t_abs : ctl->t + tfrac * ctl->dt;
        hubble_state<T>(A.H, A.bc, cell, tt, val);
    } else {
        int from[3] = {cell[0], cell[1], cell[2]};
        from[a] = A.bc[a] == 1 ? ((cell[a] % n) + n) % n : min(max(cell[a], 0), n - 1);
        const long long ps = G.pidx(from[0], from[1], from[2]);
#pragma unroll
        for (int c = 0; c < NF; ++c) val[c] = pad[c * G.fs + ps];
    }
#pragma unroll
    for (int c = 0; c < NF; ++c) pad[c * G.fs + p] = val[c];
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
// Writes the seven arrays W = (v_x, v_y, v_z, p, a_x, a_y, a_z) that the generic kernel reads.
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
        m = (double)max_speed_of_cell(u, eos, G.g[0] > 0, G.g[1] > 0, G.g[2] > 0, flag);
    }
    if (flag) ctl->flag = 1;
    block_max_to_ctl(m, ctl);
}

}  // namespace hydro
