// hydro.cu -- C ABI of libhydro_b200 (include/hydro.h): context, options, workspace carving and the
// launch sequence of one SSP-RK3 step:
//   per stage:  halo fill (a1) -> [max signal speed (a4), first CFL step only] -> stage kernels (a2-a3 of the cells
//   they read, a5-a9, and a4 of the cells stage 3 finishes); optionally replayed from a CUDA graph, or split around a
//   halo exchange for the slab decomposition
// No CPU arithmetic of the method happens here: the host only orders kernels on the caller's stream.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/hydro.h"
#include "grid.cuh"
#include "kernel_weno.cuh"
#include "kernel_generic.cuh"
#include "kernel_musta.cuh"
#include "kernels_aux.cuh"

using namespace hydro;

struct hydro_ctx {
    int n[3];
    double dx;
    int scheme, r;
    int precision = HYDRO_F64;
    int kernel = HYDRO_KERNEL_AUTO;
    int bc[3] = {HYDRO_BC_OUTFLOW, HYDRO_BC_OUTFLOW, HYDRO_BC_OUTFLOW};
    double eps = 1e-6, musta_cfl = 0.9;
    int musta_stages = 2;
    int limiter = 0;
    EosArgs eos = {0, 0.0, nullptr, 0, 0.0, 1.0};
    double t_host = 0.0;  // value to push into the control block at bind / set_option("t")
    HubbleParams H;
    cudaStream_t stream = nullptr;
    Geom G;
    // workspace
    void* ws = nullptr;
    size_t ws_bytes = 0;
    Ctl* ctl = nullptr;
    char* U[3] = {nullptr, nullptr, nullptr};  // u^n and two stage buffers (padded, 5 fields each)
    char* Wb = nullptr;                         // primitives (padded, 7 arrays) for the GENERIC kernel only (grids with an
                                                // inactive axis, "kernel" = generic), remade every stage; the marching
                                                // kernels make their primitives on the fly
    bool max_ready = false;                     // ctl->maxspeed_bits holds the max signal speed of u^n (stage-3 epilogue)
    int stage_open = 0;                         // stages of a hydro_step_stage sequence done so far (0 = between steps)
    int device = -1;                            // CUDA device of the workspace (captured at bind)
    int eos_device = -1;                        // CUDA device of the tabulated closure's table (hydro_set_eos_table)
    int zc = 0, yc = 0;                         // chunk lengths of the z / y march ("tile_zc", "sweep_zc"; 0 = default)
    bool fused_ready = false;                   // the marching kernels' shared-memory attributes are set
    char plan_err[256] = {0};
    long long launches = 0;
    // "profile" option: CUDA events around every stage-kernel launch (bench.py roofline)
    int profile = 0;
    std::vector<cudaEvent_t> ev;  // pairs (start, stop), recorded on the stream
    // "graph" option: k consecutive steady-state steps of hydro_step_cfl captured as ONE CUDA graph and replayed with
    // one cudaGraphLaunch (N4: "the whole multi-step loop in one graph"); one graph per (cfl, k), a few kept.
    struct StepGraph {
        cudaGraphExec_t exec;
        double cfl;
        int nsteps;
        long long launches;
    };
    int use_graph = 0;
    std::vector<StepGraph> graphs;
    std::string err;
};

namespace {

int fail(hydro_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        c->err = buf;
    }
    return code;
}

size_t esize(const hydro_ctx* c) { return c->precision == HYDRO_F32 ? 4 : 8; }

void make_geom(hydro_ctx* c) {
    Geom& G = c->G;
    for (int a = 0; a < 3; ++a) {
        G.n[a] = c->n[a];
        G.g[a] = c->n[a] > 1 ? c->r : 0;
        G.np[a] = G.n[a] + 2 * G.g[a];
    }
    const long long q = 16 / (long long)esize(c);  // elements per 16 bytes
    G.sx = (G.np[0] + q - 1) / q * q;
    G.sxy = G.sx * G.np[1];
    const long long vol = G.sxy * G.np[2];
    const long long q256 = 256 / (long long)esize(c);
    G.fs = (vol + q256 - 1) / q256 * q256;
}

size_t state_bytes(const hydro_ctx* c) { return (size_t)NF * (size_t)c->G.fs * esize(c); }
size_t prim_bytes(const hydro_ctx* c) { return (size_t)NW * (size_t)c->G.fs * esize(c); }
bool fused_supported(const Geom& G);
// the primitive arrays exist only where the generic kernel can be asked for
bool needs_w(const hydro_ctx* c) { return c->kernel == HYDRO_KERNEL_GENERIC || !fused_supported(c->G); }

// Every entry point that touches the device runs on the device of the workspace, whatever device is current in the
// calling thread; the caller's current device is restored on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const hydro_ctx* c) {
        if (c && c->device >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != c->device)
            switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};

#define CUDA_OK(c, call)                                                                      \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess) return fail(c, HYDRO_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

#define LAUNCHED(c, what)                                                                     \
    do {                                                                                      \
        ++(c)->launches;                                                                      \
        cudaError_t e_ = cudaGetLastError();                                                  \
        if (e_ != cudaSuccess) return fail(c, HYDRO_ECUDA, "launch %s: %s", what, cudaGetErrorString(e_)); \
    } while (0)

dim3 blk2d(int bx, int by) { return dim3(bx, by, 1); }
dim3 grd(int nx, int ny, int nz, dim3 b) { return dim3((nx + b.x - 1) / b.x, (ny + b.y - 1) / b.y, nz); }

__global__ void set_ctl_kernel(Ctl* ctl, double t, int set_t, int reset_flag) {
    if (set_t) ctl->t = t;
    if (reset_flag) {
        ctl->flag = 0;
        ctl->maxspeed_bits = 0ull;
        ctl->maxspeed_next_bits = 0ull;
        ctl->dt = 0.0;
    }
}

int need_ws(hydro_ctx* c) {
    if (!c) return HYDRO_EINVAL;
    if (!c->ws) return fail(c, HYDRO_ENOMEM, "no workspace bound (hydro_bind_workspace)");
    return HYDRO_OK;
}

template <class T>
int do_halo(hydro_ctx* c, T* pad, double tfrac, bool use_abs, double t_abs) {
    HaloArgs A;
    long long total = 0;
    for (int a = 0; a < 3; ++a) {
        A.bc[a] = c->bc[a];
        const int a1 = a == 0 ? 1 : 0, a2 = a == 2 ? 1 : 2;
        A.count[a] = c->G.g[a] ? 2LL * c->G.g[a] * c->G.n[a1] * c->G.n[a2] : 0;
        total += A.count[a];
    }
    A.H = c->H;
    A.H.dx = c->dx;
    A.eos = c->eos;
    // The closed-form Hubble ghosts are a function of ALL the Hubble axes and of the slab's own position.  Under
    // bc_z = EXTERNAL the z axis would drop out of the closed form (wrong exponent, z^2 missing from tau^2, M_z = 0),
    // the slab's z origin is not shifted, and the physical z ends would get zero-gradient planes: refused.
    if (c->bc[2] == HYDRO_BC_EXTERNAL && (c->bc[0] == HYDRO_BC_HUBBLE || c->bc[1] == HYDRO_BC_HUBBLE))
        return fail(c, HYDRO_EINVAL, "HYDRO_BC_HUBBLE on x or y cannot be combined with bc_z = HYDRO_BC_EXTERNAL "
                                     "(the slab decomposition does not carry the analytic ghost fill)");
    if (total == 0) return HYDRO_OK;
    const int tb = 256;
    halo_fill_kernel<T><<<(unsigned)((total + tb - 1) / tb), tb, 0, c->stream>>>(c->G, A, c->ctl, tfrac, t_abs,
                                                                                   use_abs ? 1 : 0, pad);
    LAUNCHED(c, "halo_fill_kernel");
    return HYDRO_OK;
}

template <class T>
int do_prim(hydro_ctx* c, const T* pad, int do_max) {
    const dim3 b = blk2d(64, 4);
    prim_kernel<T><<<grd(c->G.np[0], c->G.np[1], c->G.np[2], b), b, 0, c->stream>>>(c->G, pad, (T*)c->Wb, c->ctl,
                                                                                      do_max, c->eos);
    LAUNCHED(c, "prim_kernel");
    return HYDRO_OK;
}

template <class T>
int do_max_speed(hydro_ctx* c, const T* pad) {
    const dim3 b = blk2d(64, 4);
    max_speed_kernel<T><<<grd(c->G.n[0], c->G.n[1], c->G.n[2], b), b, 0, c->stream>>>(c->G, pad, c->ctl, c->eos);
    LAUNCHED(c, "max_speed_kernel");
    return HYDRO_OK;
}

StageArgs stage_args(const hydro_ctx* c, double ca, double cb, int mode) {
    StageArgs A;
    A.ca = ca;
    A.cb = cb;
    A.mode = mode;
    A.inv_dx = 1.0 / c->dx;
    A.eps = c->eps;
    A.musta_K = c->musta_stages;
    A.musta_C = c->musta_cfl;
    A.limiter = c->limiter;
    A.eos = c->eos;
    A.epi_max = 0;
    A.kbeg = 0;
    A.kend = c->G.n[2];
    return A;
}

// the marching kernels need all three axes active (the 400 x 1 x 1 shock tube takes the generic kernel)
bool fused_supported(const Geom& G) { return G.g[0] > 0 && G.g[1] > 0 && G.g[2] > 0; }

bool want_fused(const hydro_ctx* c) {
    if (c->kernel == HYDRO_KERNEL_GENERIC) return false;
    return fused_supported(c->G);
}

template <class T>
int configure_marching(hydro_ctx* c) {
    switch (c->scheme) {
        case HYDRO_WENO5: return configure_weno<T, 3>(c->plan_err, sizeof c->plan_err);
        case HYDRO_WENO7: return configure_weno<T, 4>(c->plan_err, sizeof c->plan_err);
        default: return configure_musta<T>(c->plan_err, sizeof c->plan_err);
    }
}

// records an event pair around the stage kernel when the "profile" option is on
struct StageTimer {
    hydro_ctx* c;
    explicit StageTimer(hydro_ctx* c_) : c(c_) {
        if (!c->profile) return;
        cudaEvent_t e0, e1;
        if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { c->profile = 0; return; }
        c->ev.push_back(e0);
        c->ev.push_back(e1);
        cudaEventRecord(e0, c->stream);
    }
    ~StageTimer() {
        if (c->profile && !c->ev.empty()) cudaEventRecord(c->ev.back(), c->stream);
    }
};

// One stage: Uout = ca u^n + cb (Us + dt L(Us)), or L(Us) itself (mode 1).
// parts / kbeg / kend (marching kernels only): bit 0 the x/z kernel over the planes [kbeg, kend), bit 1 the y sweep.
template <class T>
int do_stage(hydro_ctx* c, const T* Us, const T* Un, T* Uout, double ca, double cb, int mode, int epi_max = 0,
             int parts = 3, int kbeg = 0, int kend = -1) {
    StageArgs A = stage_args(c, ca, cb, mode);
    A.epi_max = epi_max;
    A.kbeg = kbeg;
    A.kend = kend < 0 ? c->G.n[2] : kend;
    StageTimer timer(c);
    if (want_fused(c)) {
        if (!c->fused_ready) return fail(c, HYDRO_ECUDA, "marching kernels not configured: %s", c->plan_err);
        int nl = 0, rc;
        if (c->scheme == HYDRO_MUSTA_FORCE)
            rc = launch_musta<T>(c->G, A, Us, Un, Uout, c->ctl, c->zc > 0 ? c->zc : 64, c->yc > 0 ? c->yc : 128,
                                 c->stream, parts, &nl, c->plan_err, sizeof c->plan_err);
        else {
            // default chunk lengths of the march: long chunks amortise the window priming and the one redundant flux
            // of a chunk (0.7 % at 512^3), short ones keep enough blocks in flight on small grids
            const int zc = c->zc > 0 ? c->zc : (c->G.n[2] >= 256 ? 2 * WENO_ZC : WENO_ZC);
            const int yc = c->yc > 0 ? c->yc : (c->G.n[1] >= 512 ? 2 * WENO_YC : WENO_YC);
            if (c->scheme == HYDRO_WENO5)
                rc = launch_weno<T, 3>(c->G, A, Us, Un, Uout, c->ctl, zc, yc, c->stream, parts, &nl, c->plan_err,
                                       sizeof c->plan_err);
            else
                rc = launch_weno<T, 4>(c->G, A, Us, Un, Uout, c->ctl, zc, yc, c->stream, parts, &nl, c->plan_err,
                                       sizeof c->plan_err);
        }
        if (rc != 0) return fail(c, HYDRO_ECUDA, "stage launch: %s", c->plan_err);
        c->launches += nl;
        return HYDRO_OK;
    }
    if (c->kernel == HYDRO_KERNEL_FUSED)
        return fail(c, HYDRO_EINVAL, "kernel=fused requested but the grid does not allow it (an axis is inactive)");
    const dim3 b = blk2d(32, 4);
    const dim3 g = grd(c->G.n[0], c->G.n[1], c->G.n[2], b);
    const T* W = (const T*)c->Wb;
    switch (c->scheme) {
        case HYDRO_WENO5: stage_generic_kernel<T, 0><<<g, b, 0, c->stream>>>(c->G, A, Us, W, Un, Uout, c->ctl); break;
        case HYDRO_WENO7: stage_generic_kernel<T, 1><<<g, b, 0, c->stream>>>(c->G, A, Us, W, Un, Uout, c->ctl); break;
        default: stage_generic_kernel<T, 2><<<g, b, 0, c->stream>>>(c->G, A, Us, W, Un, Uout, c->ctl); break;
    }
    LAUNCHED(c, "stage_generic_kernel");
    return HYDRO_OK;
}

// One SSP-RK3 step (a9, O8):  u1 = u + dt L(u);  u2 = 3/4 u + 1/4 (u1 + dt L(u1));
// u' = 1/3 u + 2/3 (u2 + dt L(u2)), ghosts at t, t+dt, t+dt/2.  dt_fixed > 0, or CFL mode.
// The marching kernels make con2prim + signal speeds (a2-a3) of every cell as it enters a stencil window, and stage 3
// reduces the max signal speed of the new state (a4): the max-speed pass runs as a separate kernel only for the
// first CFL step after hydro_set_state / hydro_eval_L.  Only the generic kernel reads primitive arrays (prim_kernel).
// z-halo planes of a slab (defined below)
int zhalo_impl(hydro_ctx* c, int buffer, int side, void* packed, int put);

// Overlap (slab decomposition): the planes whose z stencils stay inside the slab are launched
// first; the stream then waits for the caller's event (the neighbours' planes have arrived), the ghost planes are
// written, and the two boundary chunks and the y sweep follow.
struct Overlap {
    bool on = false;
    const void* lo = nullptr;   // packed ghost planes below / above (null: zero-gradient from the slab's own plane)
    const void* hi = nullptr;
    cudaEvent_t ready = nullptr;
};

template <class T>
int do_step_stage(hydro_ctx* c, int s, double dt_fixed, double cfl, const double* ext_max = nullptr,
                  const Overlap& ov = Overlap()) {
    T* U[3] = {(T*)c->U[0], (T*)c->U[1], (T*)c->U[2]};
    const bool weno = c->scheme != HYDRO_MUSTA_FORCE;
    const bool cflmode = !(dt_fixed > 0.0);
    const bool marching = want_fused(c);
    const double tfrac[3] = {0.0, 1.0, 0.5};
    const double ca[3] = {0.0, 0.75, 1.0 / 3.0}, cb[3] = {1.0, 0.25, 2.0 / 3.0};
    T* const in[3] = {U[0], U[1], U[2]};
    T* const out[3] = {U[1], U[2], U[0]};   // stage 3 writes u^n in place: each cell reads only its own u^n
    int rc;
    if ((rc = do_halo<T>(c, in[s], tfrac[s], false, 0.0))) return rc;
    if (ov.on && !marching) {   // generic kernel: no split; the ghost planes first (its con2prim pass reads them)
        if (ov.ready != nullptr) CUDA_OK(c, cudaStreamWaitEvent(c->stream, ov.ready, 0));
        if ((rc = zhalo_impl(c, s, 0, const_cast<void*>(ov.lo), ov.lo ? 1 : 2))) return rc;
        if ((rc = zhalo_impl(c, s, 1, const_cast<void*>(ov.hi), ov.hi ? 1 : 2))) return rc;
    }
    const bool need_max = s == 0 && cflmode && !c->max_ready && ext_max == nullptr;
    if (need_max) {   // the reduction accumulates with atomicMax: start from zero
        reset_max_kernel<<<1, 1, 0, c->stream>>>(c->ctl);
        LAUNCHED(c, "reset_max_kernel");
    }
    if (weno && !marching) {   // the generic kernel reads its primitives from arrays
        if ((rc = do_prim<T>(c, in[s], need_max ? 1 : 0))) return rc;
    } else if (need_max) {
        if ((rc = do_max_speed<T>(c, in[s]))) return rc;
    }
    if (s == 0) {
        if (ext_max != nullptr && cflmode) begin_step_ext_kernel<<<1, 1, 0, c->stream>>>(c->ctl, cfl, c->dx, ext_max);
        else begin_step_kernel<<<1, 1, 0, c->stream>>>(c->ctl, dt_fixed, cfl, c->dx);
        LAUNCHED(c, "begin_step_kernel");
        c->max_ready = false;
    }
    const int epi = (marching && s == 2) ? 1 : 0;
    if (ov.on && marching) {
        const int nz = c->G.n[2], g = c->G.g[2];
        const int b = nz >= 4 * g ? (g > 8 ? g : 8) < nz / 2 ? (g > 8 ? g : 8) : g : 0;   // planes per boundary chunk
        if (b > 0 && (rc = do_stage<T>(c, in[s], U[0], out[s], ca[s], cb[s], 0, epi, 1, b, nz - b))) return rc;
        if (ov.ready != nullptr) CUDA_OK(c, cudaStreamWaitEvent(c->stream, ov.ready, 0));
        if ((rc = zhalo_impl(c, s, 0, const_cast<void*>(ov.lo), ov.lo ? 1 : 2))) return rc;
        if ((rc = zhalo_impl(c, s, 1, const_cast<void*>(ov.hi), ov.hi ? 1 : 2))) return rc;
        if (b > 0) {
            if ((rc = do_stage<T>(c, in[s], U[0], out[s], ca[s], cb[s], 0, epi, 1, 0, b))) return rc;
            if ((rc = do_stage<T>(c, in[s], U[0], out[s], ca[s], cb[s], 0, epi, 1, nz - b, nz))) return rc;
            if ((rc = do_stage<T>(c, in[s], U[0], out[s], ca[s], cb[s], 0, epi, 2))) return rc;
        } else if ((rc = do_stage<T>(c, in[s], U[0], out[s], ca[s], cb[s], 0, epi))) return rc;
    } else if ((rc = do_stage<T>(c, in[s], U[0], out[s], ca[s], cb[s], 0, epi))) return rc;
    if (s == 2) {
        end_step_kernel<<<1, 1, 0, c->stream>>>(c->ctl);
        LAUNCHED(c, "end_step_kernel");
        c->max_ready = marching;
    }
    c->stage_open = s == 2 ? 0 : s + 1;
    return HYDRO_OK;
}

template <class T>
int do_step(hydro_ctx* c, double dt_fixed, double cfl) {
    for (int s = 0; s < 3; ++s) {
        const int rc = do_step_stage<T>(c, s, dt_fixed, cfl);
        if (rc) return rc;
    }
    return HYDRO_OK;
}

void drop_graphs(hydro_ctx* c) {
    for (auto& g : c->graphs) cudaGraphExecDestroy(g.exec);
    c->graphs.clear();
}

// A CFL step in the steady state (marching kernels, primitives and max signal speed left by the previous step's
// epilogues) is a fixed sequence of launches whose only step-dependent inputs live in the device control block:
// it can be replayed from a graph.
bool graph_ready(const hydro_ctx* c) {
    return c->use_graph && !c->profile && c->stream != nullptr && want_fused(c) && c->max_ready;
}

// Steps of one graph at most (a step is 11 kernel nodes), and graphs kept per context (the oldest is dropped).
constexpr int GRAPH_MAX_STEPS = 64;
constexpr size_t GRAPH_KEEP = 6;

template <class T>
int plain_steps(hydro_ctx* c, double cfl, int nsteps) {
    for (int s = 0; s < nsteps; ++s) {
        const int rc = do_step<T>(c, -1.0, cfl);
        if (rc) return rc;
    }
    return HYDRO_OK;
}

// nsteps (<= GRAPH_MAX_STEPS) steady-state steps with ONE cudaGraphLaunch.  Every step reads u^n from and writes
// u^{n+1} to the same buffer, and dt, t and the max signal speed live in the control block, so the k-step graph is
// the one-step sequence of nodes k times over.
template <class T>
int graph_steps(hydro_ctx* c, double cfl, int nsteps) {
    for (const auto& g : c->graphs)
        if (g.cfl == cfl && g.nsteps == nsteps) {
            CUDA_OK(c, cudaGraphLaunch(g.exec, c->stream));
            c->launches += g.launches;
            return HYDRO_OK;
        }
    // capture: nothing executes, the host-side bookkeeping of do_step is rolled back afterwards
    const long long l0 = c->launches;
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        c->use_graph = 0;   // e.g. the legacy default stream: fall back to plain launches for good
        return plain_steps<T>(c, cfl, nsteps);
    }
    const int rc = plain_steps<T>(c, cfl, nsteps);
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    hydro_ctx::StepGraph g;
    g.cfl = cfl;
    g.nsteps = nsteps;
    g.launches = c->launches - l0;
    c->launches = l0;
    if (rc != HYDRO_OK || e != cudaSuccess || graph == nullptr) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        c->use_graph = 0;
        return rc != HYDRO_OK ? rc : plain_steps<T>(c, cfl, nsteps);
    }
    const cudaError_t ei = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ei != cudaSuccess) {
        cudaGetLastError();
        c->use_graph = 0;
        return plain_steps<T>(c, cfl, nsteps);
    }
    if (c->graphs.size() >= GRAPH_KEEP) {
        cudaGraphExecDestroy(c->graphs.front().exec);
        c->graphs.erase(c->graphs.begin());
    }
    c->graphs.push_back(g);
    return graph_steps<T>(c, cfl, nsteps);
}

// z-halo planes of one state buffer <-> a packed device buffer [5][g][ny][nx] (slab decomposition, DESIGN 9).
// get: the g outermost INTERIOR planes of the side; put: the g GHOST planes of the side.
// put == 2: zero-gradient ghosts (reading Q9) made here from the slab's own boundary plane, for a slab at a physical
// outflow end of the z axis.
template <class T>
__global__ void zhalo_kernel(Geom G, T* pad, T* packed, int side, int put) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int l = blockIdx.z;   // 0 .. g-1, in increasing z
    if (i >= G.n[0] || j >= G.n[1]) return;
    const int g = G.g[2];
    const int k = put ? (side == 0 ? l - g : G.n[2] + l) : (side == 0 ? l : G.n[2] - g + l);
    const long long p = G.pidx(i, j, k);
    if (put == 2) {
        const long long ps = G.pidx(i, j, side == 0 ? 0 : G.n[2] - 1);
#pragma unroll
        for (int c = 0; c < NF; ++c) pad[c * G.fs + p] = pad[c * G.fs + ps];
        return;
    }
    const long long plane = (long long)G.n[0] * G.n[1];
    const long long q = ((long long)l * G.n[1] + j) * G.n[0] + i;
#pragma unroll
    for (int c = 0; c < NF; ++c) {
        if (put) pad[c * G.fs + p] = packed[c * g * plane + q];
        else packed[c * g * plane + q] = pad[c * G.fs + p];
    }
}

template <class T>
int eval_L_impl(hydro_ctx* c, const void* cons, double t_stage, void* L_out) {
    T* U1 = (T*)c->U[1];
    T* U2 = (T*)c->U[2];
    const dim3 b = blk2d(64, 4);
    const dim3 g = grd(c->G.n[0], c->G.n[1], c->G.n[2], b);
    int rc;
    pack_kernel<T><<<g, b, 0, c->stream>>>(c->G, (const T*)cons, U1);
    LAUNCHED(c, "pack_kernel");
    if ((rc = do_halo<T>(c, U1, 0.0, true, t_stage))) return rc;
    if (c->scheme != HYDRO_MUSTA_FORCE && !want_fused(c) && (rc = do_prim<T>(c, U1, 0))) return rc;
    if ((rc = do_stage<T>(c, U1, U1, U2, 0.0, 1.0, 1))) return rc;
    unpack_kernel<T><<<g, b, 0, c->stream>>>(c->G, U2, (T*)L_out);
    LAUNCHED(c, "unpack_kernel");
    return HYDRO_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

int hydro_create(hydro_ctx** out, int nx, int ny, int nz, double dx, int scheme) {
    if (!out || nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || scheme < 0 || scheme > 2) return HYDRO_EINVAL;
    hydro_ctx* c = new (std::nothrow) hydro_ctx;
    if (!c) return HYDRO_ENOMEM;
    c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
    c->dx = dx;
    c->scheme = scheme;
    c->r = scheme == HYDRO_WENO5 ? 3 : scheme == HYDRO_WENO7 ? 4 : 2;
    for (int a = 0; a < 3; ++a)
        if (c->n[a] > 1 && c->n[a] < c->r) { delete c; return HYDRO_EINVAL; }
    memset(&c->H, 0, sizeof c->H);
    c->H.t0 = c->H.e0 = c->H.n0 = 1.0;
    make_geom(c);
    *out = c;
    return HYDRO_OK;
}

void hydro_destroy(hydro_ctx* c) {
    if (!c) return;
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    drop_graphs(c);
    delete c;
}

const char* hydro_last_error(const hydro_ctx* c) { return c ? c->err.c_str() : "null context"; }

long long hydro_launch_count(const hydro_ctx* c) { return c ? c->launches : 0; }

int hydro_set_stream(hydro_ctx* c, void* s) {
    if (!c) return HYDRO_EINVAL;
    drop_graphs(c);
    c->stream = (cudaStream_t)s;
    return HYDRO_OK;
}

int hydro_set_option(hydro_ctx* c, const char* key, double v) {
    if (!c || !key) return HYDRO_EINVAL;
    const std::string k(key);
    drop_graphs(c);   // a captured step has the options baked into its kernel arguments
    if (k == "graph") {
        c->use_graph = v != 0.0;
    } else if (k == "precision") {
        const int p = (int)v;
        if (p != HYDRO_F64 && p != HYDRO_F32) return fail(c, HYDRO_EINVAL, "precision must be 0 or 1");
        if (c->ws && p != c->precision) return fail(c, HYDRO_EINVAL, "precision must be set before the workspace is bound");
        c->precision = p;
        make_geom(c);
    } else if (k == "kernel") {
        const int p = (int)v;
        if (p < 0 || p > 2) return fail(c, HYDRO_EINVAL, "kernel must be 0, 1 or 2");
        if (c->ws && p == HYDRO_KERNEL_GENERIC && c->Wb == nullptr)
            return fail(c, HYDRO_EINVAL, "kernel = generic needs its primitive arrays: set it before the workspace is bound");
        c->kernel = p;
    } else if (k == "tile_zc" || k == "sweep_zc") {
        if (v < 1) return fail(c, HYDRO_EINVAL, "%s < 1", key);
        (k == "tile_zc" ? c->zc : c->yc) = (int)v;
    } else if (k == "profile") {
        c->profile = v != 0.0;
    } else if (k == "bc_x" || k == "bc_y" || k == "bc_z") {
        const int b = (int)v;
        if (b < 0 || b > 3 || (b == 3 && k[3] != 'z')) return fail(c, HYDRO_EINVAL, "unknown boundary rule %d", b);
        c->bc[k[3] - 'x'] = b;
    } else if (k == "musta_stages") {
        if (v < 1) return fail(c, HYDRO_EINVAL, "musta_stages < 1");
        c->musta_stages = (int)v;
    } else if (k == "eos") {
        if (v != 0.0 && v != 1.0 && !(v == 2.0 && c->eos.tab != nullptr))
            return fail(c, HYDRO_EINVAL, "eos must be 0 (p = e/3), 1 (p = p0) or 2 (after hydro_set_eos_table)");
        c->eos.kind = (int)v;
        c->max_ready = false;   // the cached max signal speed belongs to the old closure
    } else if (k == "eos_p0") {
        if (!(v >= 0)) return fail(c, HYDRO_EINVAL, "eos_p0 < 0");
        c->eos.p0 = v;
        c->max_ready = false;
    } else if (k == "limiter") {
        if (v < 0 || v > 3) return fail(c, HYDRO_EINVAL, "limiter must be 0..3");
        c->limiter = (int)v;
    } else if (k == "musta_cfl") {
        if (!(v > 0)) return fail(c, HYDRO_EINVAL, "musta_cfl <= 0");
        c->musta_cfl = v;
    } else if (k == "weno_eps") {
        // the cross-multiplied weights take epsilon to the 4th (WENO5) or 6th (WENO7) power
        if (!(v >= 1e-40)) return fail(c, HYDRO_EINVAL, "weno_eps < 1e-40");
        c->eps = v;
    } else if (k == "t") {
        c->t_host = v;
        if (c->ws) {
            DeviceGuard dg(c);
            set_ctl_kernel<<<1, 1, 0, c->stream>>>(c->ctl, v, 1, 0);
            LAUNCHED(c, "set_ctl_kernel");
        }
    } else if (k == "x0") c->H.origin[0] = v;
    else if (k == "y0") c->H.origin[1] = v;
    else if (k == "z0") c->H.origin[2] = v;
    else if (k == "hubble_t0") c->H.t0 = v;
    else if (k == "hubble_e0") c->H.e0 = v;
    else if (k == "hubble_n0") c->H.n0 = v;
    else if (k == "hubble_bx") c->H.b[0] = v;
    else if (k == "hubble_by") c->H.b[1] = v;
    else if (k == "hubble_bz") c->H.b[2] = v;
    else return fail(c, HYDRO_EINVAL, "unknown option '%s'", key);
    return HYDRO_OK;
}

size_t hydro_workspace_bytes(const hydro_ctx* c) {
    if (!c) return 0;
    return 256 + 3 * state_bytes(c) + (needs_w(c) ? prim_bytes(c) : 0);  // control block, U0, U1, U2, [W]
}

int hydro_bind_workspace(hydro_ctx* c, void* p, size_t bytes) {
    if (!c || !p) return HYDRO_EINVAL;
    if (((size_t)p & 255) != 0) return fail(c, HYDRO_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < hydro_workspace_bytes(c))
        return fail(c, HYDRO_ENOMEM, "workspace too small: %zu < %zu", bytes, hydro_workspace_bytes(c));
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, p) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return fail(c, HYDRO_EINVAL, "workspace is not CUDA device memory");
    }
    if (c->eos.tab != nullptr && c->eos_device != attr.device)
        return fail(c, HYDRO_EINVAL, "workspace on GPU %d, equation-of-state table on GPU %d", attr.device, c->eos_device);
    c->device = attr.device;
    DeviceGuard dg(c);
    c->ws = p;
    c->ws_bytes = bytes;
    char* base = (char*)p;
    c->ctl = (Ctl*)base;
    const size_t sb = state_bytes(c);
    for (int i = 0; i < 3; ++i) c->U[i] = base + 256 + i * sb;
    c->Wb = needs_w(c) ? base + 256 + 3 * sb : nullptr;
    c->max_ready = false;
    c->stage_open = 0;
    drop_graphs(c);
    CUDA_OK(c, cudaMemsetAsync(p, 0, hydro_workspace_bytes(c), c->stream));
    set_ctl_kernel<<<1, 1, 0, c->stream>>>(c->ctl, c->t_host, 1, 1);
    LAUNCHED(c, "set_ctl_kernel");
    c->fused_ready = false;
    if (fused_supported(c->G)) {
        c->fused_ready = (c->precision == HYDRO_F64 ? configure_marching<double>(c) : configure_marching<float>(c)) == 0;
        if (!c->fused_ready && c->kernel != HYDRO_KERNEL_GENERIC)
            return fail(c, HYDRO_ECUDA, "marching kernels: %s", c->plan_err);
    }
    return HYDRO_OK;
}

int hydro_set_state(hydro_ctx* c, const void* cons) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!cons) return HYDRO_EINVAL;
    const dim3 b = blk2d(64, 4);
    const dim3 g = grd(c->G.n[0], c->G.n[1], c->G.n[2], b);
    if (c->precision == HYDRO_F64) pack_kernel<double><<<g, b, 0, c->stream>>>(c->G, (const double*)cons, (double*)c->U[0]);
    else pack_kernel<float><<<g, b, 0, c->stream>>>(c->G, (const float*)cons, (float*)c->U[0]);
    LAUNCHED(c, "pack_kernel");
    c->max_ready = false;
    c->stage_open = 0;
    set_ctl_kernel<<<1, 1, 0, c->stream>>>(c->ctl, 0.0, 0, 1);   // the time is the caller's ("t" option): kept
    LAUNCHED(c, "set_ctl_kernel");
    return HYDRO_OK;
}

int hydro_get_state(hydro_ctx* c, void* out) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!out) return HYDRO_EINVAL;
    const dim3 b = blk2d(64, 4);
    const dim3 g = grd(c->G.n[0], c->G.n[1], c->G.n[2], b);
    if (c->precision == HYDRO_F64) unpack_kernel<double><<<g, b, 0, c->stream>>>(c->G, (const double*)c->U[0], (double*)out);
    else unpack_kernel<float><<<g, b, 0, c->stream>>>(c->G, (const float*)c->U[0], (float*)out);
    LAUNCHED(c, "unpack_kernel");
    return HYDRO_OK;
}

// Host entry points: stage through the third state buffer, which is idle BETWEEN steps (inside a
// hydro_step_stage sequence it is a live stage input, so the calls are refused there).
int hydro_set_state_host(hydro_ctx* c, const void* cons_host) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!cons_host) return HYDRO_EINVAL;
    if (c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_set_state_host inside a hydro_step_stage sequence");
    const size_t bytes = (size_t)NF * c->n[0] * c->n[1] * c->n[2] * esize(c);
    CUDA_OK(c, cudaMemcpyAsync(c->U[2], cons_host, bytes, cudaMemcpyHostToDevice, c->stream));
    if ((rc = hydro_set_state(c, c->U[2]))) return rc;
    CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return HYDRO_OK;
}

int hydro_get_state_host(hydro_ctx* c, void* out_host) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!out_host) return HYDRO_EINVAL;
    if (c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_get_state_host inside a hydro_step_stage sequence");
    const size_t bytes = (size_t)NF * c->n[0] * c->n[1] * c->n[2] * esize(c);
    if ((rc = hydro_get_state(c, c->U[2]))) return rc;
    CUDA_OK(c, cudaMemcpyAsync(out_host, c->U[2], bytes, cudaMemcpyDeviceToHost, c->stream));
    CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return HYDRO_OK;
}

int hydro_step(hydro_ctx* c, double dt, int nsteps) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!(dt > 0) || nsteps < 0) return fail(c, HYDRO_EINVAL, "hydro_step: dt <= 0 or nsteps < 0");
    if (c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_step inside a hydro_step_stage sequence");
    for (int s = 0; s < nsteps; ++s) {
        rc = c->precision == HYDRO_F64 ? do_step<double>(c, dt, 0.0) : do_step<float>(c, dt, 0.0);
        if (rc) return rc;
    }
    return HYDRO_OK;
}

int hydro_step_cfl(hydro_ctx* c, double cfl, int nsteps) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!(cfl > 0) || nsteps < 0) return fail(c, HYDRO_EINVAL, "hydro_step_cfl: cfl <= 0 or nsteps < 0");
    if (c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_step_cfl inside a hydro_step_stage sequence");
    for (int s = 0; s < nsteps;) {
        int k = 1;
        if (graph_ready(c)) {   // all the steps that are left (in pieces of GRAPH_MAX_STEPS) from one graph launch each
            k = nsteps - s < GRAPH_MAX_STEPS ? nsteps - s : GRAPH_MAX_STEPS;
            rc = c->precision == HYDRO_F64 ? graph_steps<double>(c, cfl, k) : graph_steps<float>(c, cfl, k);
        } else rc = c->precision == HYDRO_F64 ? do_step<double>(c, -1.0, cfl) : do_step<float>(c, -1.0, cfl);
        if (rc) return rc;
        s += k;
    }
    return HYDRO_OK;
}

int hydro_set_eos_table(hydro_ctx* c, const void* p_device, int n, double e_min, double e_max) {
    if (!c) return HYDRO_EINVAL;
    if (!p_device || n < 2 || !(e_max > e_min)) return fail(c, HYDRO_EINVAL, "hydro_set_eos_table: null table, n < 2 or e_max <= e_min");
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, p_device) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        cudaGetLastError();
        return fail(c, HYDRO_EINVAL, "hydro_set_eos_table: the table is not CUDA device memory");
    }
    if (c->ws != nullptr && attr.device != c->device)
        return fail(c, HYDRO_EINVAL, "hydro_set_eos_table: the table is on GPU %d, the workspace on GPU %d", attr.device, c->device);
    drop_graphs(c);
    c->eos_device = attr.device;
    c->eos.tab = (const double*)p_device;
    c->eos.n = n;
    c->eos.e_min = e_min;
    c->eos.de = (e_max - e_min) / (n - 1);
    c->eos.kind = 2;
    c->max_ready = false;
    return HYDRO_OK;
}

int hydro_step_cfl_batch(hydro_ctx** ctxs, int nctx, double cfl, int nsteps) {
    if (!ctxs || nctx < 0) return HYDRO_EINVAL;
    for (int i = 0; i < nctx; ++i)
        if (!ctxs[i]) return HYDRO_EINVAL;
    // step by step over the batch, so that the launches of the contexts interleave on their streams; once every
    // context can replay from a graph, each gets all its remaining steps at once (one graph launch per context)
    for (int s = 0; s < nsteps; ++s) {
        bool all_graph = nctx > 0;
        for (int i = 0; i < nctx; ++i) all_graph = all_graph && graph_ready(ctxs[i]);
        for (int i = 0; i < nctx; ++i) {
            const int rc = hydro_step_cfl(ctxs[i], cfl, all_graph ? nsteps - s : 1);
            if (rc) return rc;
        }
        if (all_graph) break;
    }
    return HYDRO_OK;
}

int hydro_max_signal_speed(hydro_ctx* c, double* out_host) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!out_host) return HYDRO_EINVAL;
    if (c->max_ready) {   // the stage-3 epilogue of the last step left the max speed of u^n in the control block
        Ctl h0;
        CUDA_OK(c, cudaMemcpyAsync(&h0, c->ctl, sizeof h0, cudaMemcpyDeviceToHost, c->stream));
        CUDA_OK(c, cudaStreamSynchronize(c->stream));
        if (h0.maxspeed_bits != 0ull) {
            memcpy(out_host, &h0.maxspeed_bits, sizeof(double));
            return HYDRO_OK;
        }
    }
    reset_max_kernel<<<1, 1, 0, c->stream>>>(c->ctl);
    LAUNCHED(c, "reset_max_kernel");
    rc = c->precision == HYDRO_F64 ? do_max_speed<double>(c, (const double*)c->U[0])
                                   : do_max_speed<float>(c, (const float*)c->U[0]);
    if (rc) return rc;
    Ctl h;
    CUDA_OK(c, cudaMemcpyAsync(&h, c->ctl, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    CUDA_OK(c, cudaStreamSynchronize(c->stream));
    memcpy(out_host, &h.maxspeed_bits, sizeof(double));
    // the value stays in the control block: it is the max speed of u^n, which is what the next CFL step needs
    c->max_ready = true;
    return HYDRO_OK;
}

int hydro_eval_L(hydro_ctx* c, const void* cons, double t_stage, void* L_out) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!cons || !L_out) return HYDRO_EINVAL;
    if (c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_eval_L inside a hydro_step_stage sequence");
    return c->precision == HYDRO_F64 ? eval_L_impl<double>(c, cons, t_stage, L_out)
                                     : eval_L_impl<float>(c, cons, t_stage, L_out);
}

size_t hydro_zhalo_elems(const hydro_ctx* c) {
    if (!c) return 0;
    return (size_t)NF * c->G.g[2] * c->G.n[1] * c->G.n[0];
}

}  // extern "C"
namespace {
int zhalo_impl(hydro_ctx* c, int buffer, int side, void* packed, int put) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if ((!packed && put != 2) || buffer < 0 || buffer > 2 || (side != 0 && side != 1))
        return fail(c, HYDRO_EINVAL, "zhalo: bad argument");
    if (c->G.g[2] == 0) return fail(c, HYDRO_EINVAL, "zhalo: the z axis is inactive");
    const dim3 b = blk2d(64, 4);
    const dim3 g((c->G.n[0] + b.x - 1) / b.x, (c->G.n[1] + b.y - 1) / b.y, c->G.g[2]);
    if (c->precision == HYDRO_F64) zhalo_kernel<double><<<g, b, 0, c->stream>>>(c->G, (double*)c->U[buffer], (double*)packed, side, put);
    else zhalo_kernel<float><<<g, b, 0, c->stream>>>(c->G, (float*)c->U[buffer], (float*)packed, side, put);
    LAUNCHED(c, "zhalo_kernel");
    return HYDRO_OK;
}
}  // namespace
extern "C" {
int hydro_get_zhalo(hydro_ctx* c, int buffer, int side, void* packed_out) { return zhalo_impl(c, buffer, side, packed_out, 0); }
int hydro_put_zhalo(hydro_ctx* c, int buffer, int side, const void* packed_in) {
    return zhalo_impl(c, buffer, side, const_cast<void*>(packed_in), packed_in ? 1 : 2);
}

int hydro_step_stage(hydro_ctx* c, double dt, int stage) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!(dt > 0) || stage < 0 || stage > 2) return fail(c, HYDRO_EINVAL, "hydro_step_stage: dt <= 0 or stage not in 0..2");
    if (stage != c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_step_stage: stage %d out of order (expected %d)", stage, c->stage_open);
    return c->precision == HYDRO_F64 ? do_step_stage<double>(c, stage, dt, 0.0) : do_step_stage<float>(c, stage, dt, 0.0);
}

int hydro_step_stage_cfl(hydro_ctx* c, double cfl, int stage, const void* maxspeed_dev) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!(cfl > 0) || stage < 0 || stage > 2 || !maxspeed_dev)
        return fail(c, HYDRO_EINVAL, "hydro_step_stage_cfl: cfl <= 0, stage not in 0..2 or null pointer");
    if (stage != c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_step_stage_cfl: stage %d out of order (expected %d)", stage, c->stage_open);
    const double* m = (const double*)maxspeed_dev;
    return c->precision == HYDRO_F64 ? do_step_stage<double>(c, stage, -1.0, cfl, m) : do_step_stage<float>(c, stage, -1.0, cfl, m);
}

int hydro_step_stage_overlap(hydro_ctx* c, double cfl, int stage, const void* maxspeed_dev, const void* ghosts_lo_dev,
                             const void* ghosts_hi_dev, void* ready_event) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!(cfl > 0) || stage < 0 || stage > 2 || !maxspeed_dev)
        return fail(c, HYDRO_EINVAL, "hydro_step_stage_overlap: cfl <= 0, stage not in 0..2 or null pointer");
    if (c->bc[2] != HYDRO_BC_EXTERNAL || c->G.g[2] == 0)
        return fail(c, HYDRO_EINVAL, "hydro_step_stage_overlap needs bc_z = HYDRO_BC_EXTERNAL on an active z axis");
    if (stage != c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_step_stage_overlap: stage %d out of order (expected %d)", stage, c->stage_open);
    Overlap ov;
    ov.on = true;
    ov.lo = ghosts_lo_dev;
    ov.hi = ghosts_hi_dev;
    ov.ready = (cudaEvent_t)ready_event;
    const double* m = (const double*)maxspeed_dev;
    return c->precision == HYDRO_F64 ? do_step_stage<double>(c, stage, -1.0, cfl, m, ov)
                                     : do_step_stage<float>(c, stage, -1.0, cfl, m, ov);
}

int hydro_local_max_speed(hydro_ctx* c, void* maxspeed_dev_out) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!maxspeed_dev_out) return HYDRO_EINVAL;
    if (c->stage_open) return fail(c, HYDRO_EINVAL, "hydro_local_max_speed inside a hydro_step_stage sequence");
    if (!c->max_ready) {
        reset_max_kernel<<<1, 1, 0, c->stream>>>(c->ctl);
        LAUNCHED(c, "reset_max_kernel");
        rc = c->precision == HYDRO_F64 ? do_max_speed<double>(c, (const double*)c->U[0])
                                       : do_max_speed<float>(c, (const float*)c->U[0]);
        if (rc) return rc;
        c->max_ready = true;
    }
    // the control block keeps the max as the bit pattern of a non-negative double: the 8 bytes ARE the double
    CUDA_OK(c, cudaMemcpyAsync(maxspeed_dev_out, &c->ctl->maxspeed_bits, sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    return HYDRO_OK;
}

int hydro_stage_kernel_time(hydro_ctx* c, double* ms_total_host, long long* launches_host) {
    if (!c || !ms_total_host || !launches_host) return HYDRO_EINVAL;
    CUDA_OK(c, cudaStreamSynchronize(c->stream));
    double total = 0.0;
    for (size_t i = 0; i + 1 < c->ev.size(); i += 2) {
        float ms = 0.f;
        CUDA_OK(c, cudaEventElapsedTime(&ms, c->ev[i], c->ev[i + 1]));
        total += ms;
    }
    *ms_total_host = total;
    *launches_host = (long long)(c->ev.size() / 2);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    c->ev.clear();
    return HYDRO_OK;
}

int hydro_get_time(hydro_ctx* c, double* t_host) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    if (!t_host) return HYDRO_EINVAL;
    Ctl h;
    CUDA_OK(c, cudaMemcpyAsync(&h, c->ctl, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    CUDA_OK(c, cudaStreamSynchronize(c->stream));
    *t_host = h.t;
    return HYDRO_OK;
}

int hydro_status(hydro_ctx* c) {
    int rc = need_ws(c);
    if (rc) return rc;
    DeviceGuard dg(c);
    Ctl h;
    CUDA_OK(c, cudaMemcpyAsync(&h, c->ctl, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    CUDA_OK(c, cudaStreamSynchronize(c->stream));
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(c, HYDRO_ECUDA, "%s", cudaGetErrorString(e));
    return h.flag ? fail(c, HYDRO_EUNPHYSICAL, "con2prim clamped at least one cell") : HYDRO_OK;
}

}  // extern "C"

// ================================================================================================
// hydro_max_signal_speed_static -- the max signal speed (a3-a4) for callers that may not allocate device memory.
//
// Everything above works in memory the caller hands over (hydro_bind_workspace); the reduction of
// hydro_max_signal_speed keeps its accumulator in that workspace.  Some callers have no workspace to give and cannot
// get one: a monitoring or time-step hook that runs inside someone else's event loop and is handed a state it does
// not own, a process whose device memory is wholly owned by a framework's pool that is already at its cap, or a
// latency-bound loop in which cudaMalloc is off limits because it synchronises the whole device and would stall the
// other events' streams.  For them this entry point reduces in a fixed array that is part of the library's own
// image: `static_scratch` below, 256 B of header + one double per tile of 64 x 4 x 1 cells, 512.25 KiB in all.
// Every GPU that loads the library holds that array until the process exits, which is why it is kept small; the price
// is the size limit STATIC_MAX_TILES (256^3 is the largest cube).
//
// Variant of max_speed_kernel: the same per-cell function, but every block stores the maximum of its tile in the
// scratch array and takes a ticket; the block that draws the last ticket reduces the tiles' values, writes the
// caller's output and puts the ticket counter back to zero.  No atomics on doubles, no workspace, no control block.
namespace {

constexpr unsigned STATIC_TILE_X = 64, STATIC_TILE_Y = 4;
constexpr unsigned STATIC_MAX_TILES = 65536;
constexpr size_t STATIC_HEAD = 256;   // [0] ticket counter (unsigned), rest unused
constexpr size_t STATIC_BYTES = STATIC_HEAD + (size_t)STATIC_MAX_TILES * sizeof(double);

// In host code this name is only a handle for cudaGetSymbolAddress (a kernel given `static_scratch` itself would be
// given a host address); static_scratch_on() below turns it into the array's address on one device.
static __device__ __align__(256) unsigned char static_scratch[STATIC_BYTES];

// block-wide max of a non-negative value; the result is valid in thread 0
__device__ __forceinline__ double block_max_static(double m, double* smax) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    const int tid = threadIdx.x;
    __syncthreads();   // smax may still be read from a previous use
    if ((tid & 31) == 0) smax[tid >> 5] = m;
    __syncthreads();
    if (tid < 32) {
        m = tid < (int)(blockDim.x >> 5) ? smax[tid] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    }
    return m;
}

// cons: the caller's INTERIOR state [5][nz][ny][nx] (no ghosts, no padding).  One block of 256 threads per tile;
// tiles numbered x fastest, then y, then z.
template <class T>
__global__ void __launch_bounds__(256) max_speed_static_kernel(int nx, int ny, int nz, unsigned tiles_x, unsigned tiles_y,
                                                               const T* __restrict__ cons, EosArgs eos,
                                                               unsigned char* scratch, double* __restrict__ out) {
    __shared__ double smax[8];
    __shared__ bool last;
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch);
    double* tile_max = reinterpret_cast<double*>(scratch + STATIC_HEAD);
    const unsigned tile = blockIdx.x, ntiles = gridDim.x;
    const unsigned bx = tile % tiles_x, by = (tile / tiles_x) % tiles_y;
    const int k = (int)(tile / (tiles_x * tiles_y));
    const int i = (int)(bx * STATIC_TILE_X + (threadIdx.x % STATIC_TILE_X));
    const int j = (int)(by * STATIC_TILE_Y + (threadIdx.x / STATIC_TILE_X));
    double m = 0.0;
    if (i < nx && j < ny) {
        const long long N = (long long)nx * ny * nz;
        const long long q = ((long long)k * ny + j) * nx + i;
        const T u[NF] = {cons[q], cons[N + q], cons[2 * N + q], cons[3 * N + q], (T)0};
        int flag = 0;   // a clamped cell enters with its clamped speed; this call has no status word to raise
        m = (double)max_speed_of_cell(u, eos, nx > 1, ny > 1, nz > 1, flag);
    }
    m = block_max_static(m, smax);
    if (threadIdx.x == 0) {
        tile_max[tile] = m;
        __threadfence();   // the tile's value is visible before the ticket is
        last = atomicAdd(ticket, 1u) == ntiles - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double r = 0.0;
    for (unsigned b = threadIdx.x; b < ntiles; b += blockDim.x) r = fmax(r, __ldcg(tile_max + b));
    r = block_max_static(r, smax);
    if (threadIdx.x == 0) {
        *out = r;
        *ticket = 0u;   // the next call on this device starts from zero again
    }
}

// Address of static_scratch on `device`, which must be the current device.  Looked up once per device.
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex static_mu;
unsigned char* static_ptr[STATIC_MAX_DEVICES] = {};

cudaError_t static_scratch_on(int device, unsigned char** p) {
    std::lock_guard<std::mutex> lock(static_mu);
    if (static_ptr[device] == nullptr) {
        void* a = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&a, static_scratch);
        if (e != cudaSuccess) return e;
        static_ptr[device] = static_cast<unsigned char*>(a);
    }
    *p = static_ptr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" int hydro_max_signal_speed_static(hydro_ctx* c, const void* cons_device, void* maxspeed_device_out) {
    if (!c) return HYDRO_EINVAL;
    if (!cons_device || !maxspeed_device_out) return fail(c, HYDRO_EINVAL, "hydro_max_signal_speed_static: null pointer");
    const unsigned long long tx = ((unsigned)c->n[0] + STATIC_TILE_X - 1) / STATIC_TILE_X;
    const unsigned long long ty = ((unsigned)c->n[1] + STATIC_TILE_Y - 1) / STATIC_TILE_Y;
    const unsigned long long tiles = tx * ty * (unsigned long long)c->n[2];
    if (tiles > STATIC_MAX_TILES)
        return fail(c, HYDRO_EINVAL,
                    "hydro_max_signal_speed_static: a %d x %d x %d grid is %llu tiles of %u x %u x 1 cells, the built-in "
                    "scratch array holds %u (e.g. 256^3); use hydro_max_signal_speed with a workspace",
                    c->n[0], c->n[1], c->n[2], tiles, STATIC_TILE_X, STATIC_TILE_Y, STATIC_MAX_TILES);
    cudaPointerAttributes ai, ao;
    if (cudaPointerGetAttributes(&ai, cons_device) != cudaSuccess || ai.type != cudaMemoryTypeDevice ||
        cudaPointerGetAttributes(&ao, maxspeed_device_out) != cudaSuccess || ao.type != cudaMemoryTypeDevice ||
        ai.device != ao.device) {
        cudaGetLastError();
        return fail(c, HYDRO_EINVAL, "hydro_max_signal_speed_static: state and output must be CUDA device memory of one GPU");
    }
    const int dev = ai.device;
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(c, HYDRO_EINVAL, "hydro_max_signal_speed_static: device %d", dev);
    // run on the device that holds the state; the caller's current device is put back on return
    int prev = -1;
    CUDA_OK(c, cudaGetDevice(&prev));
    struct Back {
        int prev, dev;
        ~Back() { if (prev != dev) cudaSetDevice(prev); }
    } back{prev, dev};
    if (prev != dev) CUDA_OK(c, cudaSetDevice(dev));
    unsigned char* scratch = nullptr;
    CUDA_OK(c, static_scratch_on(dev, &scratch));
    // the ticket counter must start at zero even if an earlier call on this device never finished
    CUDA_OK(c, cudaMemsetAsync(scratch, 0, STATIC_HEAD, c->stream));
    if (c->precision == HYDRO_F64)
        max_speed_static_kernel<double><<<(unsigned)tiles, 256, 0, c->stream>>>(
            c->n[0], c->n[1], c->n[2], (unsigned)tx, (unsigned)ty, (const double*)cons_device, c->eos, scratch,
            (double*)maxspeed_device_out);
    else
        max_speed_static_kernel<float><<<(unsigned)tiles, 256, 0, c->stream>>>(
            c->n[0], c->n[1], c->n[2], (unsigned)tx, (unsigned)ty, (const float*)cons_device, c->eos, scratch,
            (double*)maxspeed_device_out);
    LAUNCHED(c, "max_speed_static_kernel");
    return HYDRO_OK;
}
