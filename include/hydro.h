/* hydro.h -- C ABI of libhydro_b200: the data-parallel hot path of arxiv 1604.03360
 * ("Relativistic hydrodynamics on graphics processing units") on NVIDIA B200 (sm_100a).
 *
 * What the library computes (citations are PAPER.md lines, i.e. the paper's text):
 *   - the conservative system of Eq. (1), for five fields E, M_x, M_y, M_z, R
 *     (energy, momenta, conserved charge) with the equation of state p = e/3;
 *   - the method-of-lines operator L(u) of Eq. (2): for every cell the sum over the
 *     active axes of (f(x - e_i/2) - f(x + e_i/2)) / |e_i| with interface fluxes from
 *       WENO5 / WENO7 finite-difference reconstruction (section 1.2) on local
 *       Lax-Friedrichs split fluxes, or
 *       MUSTA-FORCE with MUSCL/minmod (section 1.1);
 *   - the "standard, third order Runge-Kutta" of PAPER.md:20 (Shu-Osher SSP-RK3): three L(u) per step.
 * Everything the paper does not print (EOS, splitting, wave speeds, epsilon, ghost rules) follows the
 * readings Q1..Q18 listed in DESIGN.md section 3.
 *
 * Conventions
 *   - Every function returns a status (HYDRO_OK = 0 or a negative HYDRO_E*); nothing throws or aborts.
 *     hydro_last_error() gives a text for the last failure on that context.
 *   - "device pointer" = CUDA device memory owned by the caller (e.g. torch.empty(..., device="cuda")
 *     .data_ptr()); "host pointer" = ordinary host memory owned by the caller.  The library never frees
 *     or keeps a caller buffer beyond the call, except the workspace bound with hydro_bind_workspace,
 *     which must stay alive until hydro_destroy or the next bind.
 *   - State layout at the boundary: interior cells only, [5][nz][ny][nx], x fastest, field order
 *     E, M_x, M_y, M_z, R; element type double (HYDRO_F64) or float (HYDRO_F32) per "precision".
 *     Ghost cells are internal to the library.
 *   - An axis with n = 1 is inactive: no sweep, no ghosts, not part of the max signal speed.  This is
 *     how the 1+1D shock tube runs as 400 x 1 x 1.
 *   - All work is enqueued on the stream set with hydro_set_stream (default: the legacy default
 *     stream).  Calls that return data to the host synchronise that stream; the others are
 *     asynchronous.  One context per stream; a context is not thread-safe.
 *   - There is no CPU fallback anywhere: without a CUDA device every compute call fails with
 *     HYDRO_ECUDA.
 */
#ifndef HYDRO_B200_H
#define HYDRO_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hydro_ctx hydro_ctx; /* opaque, owned by the library */

enum { HYDRO_WENO5 = 0, HYDRO_WENO7 = 1, HYDRO_MUSTA_FORCE = 2 };          /* scheme            */
enum { HYDRO_BC_OUTFLOW = 0, HYDRO_BC_PERIODIC = 1, HYDRO_BC_HUBBLE = 2,
       HYDRO_BC_EXTERNAL = 3 /* z only: the caller provides the ghost planes (hydro_put_zhalo) */ }; /* per axis */
enum { HYDRO_F64 = 0, HYDRO_F32 = 1 };                                     /* "precision"       */
enum { HYDRO_KERNEL_AUTO = 0, HYDRO_KERNEL_GENERIC = 1, HYDRO_KERNEL_FUSED = 2 }; /* "kernel"   */
enum {
    HYDRO_OK = 0,
    HYDRO_EINVAL = -1,      /* bad argument, unknown option, call out of order                   */
    HYDRO_ENOMEM = -2,      /* workspace missing or too small                                    */
    HYDRO_ECUDA = -3,       /* a CUDA runtime call or kernel launch failed (text in last_error)  */
    HYDRO_EUNPHYSICAL = -4  /* con2prim had to clamp a cell (E < 1e-300, |M| > (1-1e-12) E) or met a
                               non-finite value (NaN / Inf energy or momentum)                  */
};

/* Create a context for an nx x ny x nz grid of spacing dx (same on all axes, the |e_i| of Eq. (2),
 * PAPER.md:17-20) and one of the three schemes.  Allocates no device memory.  Ghost width on active
 * axes: 3 (WENO5), 4 (WENO7), 2 (MUSTA-FORCE).  EINVAL for n < 1, dx <= 0, unknown scheme, or an
 * active axis shorter than the ghost width. */
int hydro_create(hydro_ctx **out, int nx, int ny, int nz, double dx, int scheme);

/* Set an option.  "precision" and "kernel" = HYDRO_KERNEL_GENERIC must precede hydro_bind_workspace (both change the
 * workspace size; EINVAL afterwards).
 *   "precision"     HYDRO_F64 (default) | HYDRO_F32: arithmetic and storage type of the whole path
 *   "bc_x|bc_y|bc_z" boundary rule per axis (default outflow = copy the nearest interior cell)
 *   "weno_eps"      epsilon of the WENO weights (default 1e-6, reading Q5; EINVAL below 1e-40: the weights are
 *                   evaluated cross-multiplied, which takes epsilon to the 6th power.  For the same reason fp64
 *                   data must stay below about 1e25 in magnitude.  The fp32 path rescales its indicators by a power of
 *                   two, so its bound is the plain overflow of the indicators themselves (squares of flux
 *                   differences, with coefficients of order 1e4 in WENO7): fp32 conserved values must stay below
 *                   about 1e16 for WENO5 and 1e13 for WENO7; beyond that L(u) is not finite)
 *   "musta_stages"  K of MUSTA-FORCE (default 2, reading Q8);  "musta_cfl" its local Courant number
 *                   (default 0.9, reading Q7)
 *   "eos", "eos_p0" equation of state: 0 (default) p = e/3 (reading Q2); 1 p = eos_p0, a constant (the closure for
 *                   which the free-streaming flow of the paper's ref. [8] is exact, reading Q14); the
 *                   characteristic speeds are then all v_d
 *   "limiter"       MUSCL slope limiter of MUSTA-FORCE: 0 minmod (default, reading Q6), 1 van Leer, 2 MC,
 *                   3 superbee ("a variety of slope limiting methods")
 *   "t"             current time (used by the analytic Hubble ghost fill)
 *   "x0|y0|z0"      coordinate of the low face of the domain on each axis
 *   "hubble_t0|hubble_e0|hubble_n0|hubble_bx|hubble_by|hubble_bz"  parameters of the closed-form
 *                   Hubble flow used by HYDRO_BC_HUBBLE (readings Q13, Q14)
 *   "tile_zc", "sweep_zc"  cells a block of the x/z kernel marches through along z / of the y sweep along y
 *                   (defaults 64 / 128 for all kernels, doubled for the WENO kernels on axes of 256 / 512 cells or more; tuning knobs: a longer
 *                   march amortises the one redundant flux and the pipeline fill of a chunk)
 *   "profile"       0 (default) | 1: record a CUDA event pair on the stream around every stage-kernel
 *                   launch, read back with hydro_stage_kernel_time
 *   "graph"         0 (default) | 1: hydro_step_cfl(ctx, cfl, k) replays its k steady-state steps from ONE CUDA graph
 *                   (one cudaGraphLaunch instead of 11 k kernel launches, in pieces of at most 64 steps; every
 *                   step-dependent value, dt included, lives in the device control block; one graph per (cfl, k), the
 *                   six most recent are kept).  hydro_step_cfl_batch gives each context all its steps in one launch
 *                   once every context of the batch can replay.  Needs a non-default stream (hydro_set_stream) and the
 *                   marching kernels; on the legacy default stream, with "profile" on, or while the control block
 *                   does not yet hold the max signal speed of u^n (i.e. before the stage-3 epilogue of a first plain
 *                   step, or hydro_max_signal_speed, has left it there) the plain launches run instead.  The
 *                   graphs are dropped whenever an option, the stream or the workspace changes.
 *   "kernel"        HYDRO_KERNEL_AUTO (default: the marching stage kernels where all three axes are active,
 *                   else the generic one-thread-per-cell kernel) | HYDRO_KERNEL_GENERIC | HYDRO_KERNEL_FUSED
 *                   (= marching; EINVAL at step time if the grid does not allow it)
 * EINVAL for an unknown key or a value out of range. */
int hydro_set_option(hydro_ctx *ctx, const char *key, double value);

/* cuda_stream: a cudaStream_t passed as void* (torch.cuda.current_stream().cuda_stream); NULL = the
 * legacy default stream. */
int hydro_set_stream(hydro_ctx *ctx, void *cuda_stream);

/* Bytes of device memory the context needs: a 256-byte control block and three padded states (u^n and two RK stage
 * buffers, five arrays each).  The marching kernels make their primitives on the fly and keep none in memory; only
 * where the generic kernel can run ("kernel" = HYDRO_KERNEL_GENERIC, or a grid with an inactive axis) ONE set of the
 * seven per-cell primitive arrays (v_x, v_y, v_z, p, a_x, a_y, a_z) is added.  Depends on "precision" and "kernel". */
size_t hydro_workspace_bytes(const hydro_ctx *ctx);

/* Hand the context its device memory (256-byte aligned, at least hydro_workspace_bytes()).  The caller
 * keeps ownership.  ENOMEM if too small, EINVAL if misaligned or not CUDA device memory.  Zero-fills it on the
 * stream.  The context remembers the device the memory lives on: every later call runs there whatever device is
 * current in the calling thread (and restores the caller's current device before returning). */
int hydro_bind_workspace(hydro_ctx *ctx, void *device_ptr, size_t bytes);

/* Copy the interior conserved state in from / out to a DEVICE pointer ([5][nz][ny][nx], element type
 * per "precision").  Asynchronous on the stream.  set_state also clears the unphysical flag and the cached max
 * signal speed; the current time is NOT touched (it only changes through the "t" option and by stepping). */
int hydro_set_state(hydro_ctx *ctx, const void *cons_device);
int hydro_get_state(hydro_ctx *ctx, void *cons_device_out);

/* The same through HOST pointers: the library stages through its third state buffer (idle between steps) with
 * cudaMemcpyAsync and synchronises the stream before returning.  These are the end-to-end entry points
 * (bench.py "e2e").  EINVAL between hydro_step_stage(., 0) and hydro_step_stage(., 2), where that buffer is live. */
int hydro_set_state_host(hydro_ctx *ctx, const void *cons_host);
int hydro_get_state_host(hydro_ctx *ctx, void *cons_host_out);

/* Advance nsteps SSP-RK3 steps of fixed size dt (per stage: ghost fill, con2prim +
 * signal speeds, L(u) of Eq. (2) fused with the Runge-Kutta combination).  Asynchronous. */
int hydro_step(hydro_ctx *ctx, double dt, int nsteps);

/* The same with dt = cfl * dx / (max signal speed of the state at the start of each step), the maximum taken on the
 * device: by the stage-3 epilogue of the previous step's y sweep (marching kernels), else by a reduction pass before
 * stage 1 (first step after hydro_set_state, generic kernel).  No host synchronisation (reading Q10).  Asynchronous. */
int hydro_step_cfl(hydro_ctx *ctx, double cfl, int nsteps);

/* Tabulated barotropic equation of state p(e) (the quark-gluon-plasma physics the solver
 * is for needs a general equation of state): n >= 2 values p(e_i) at e_i = e_min + i (e_max - e_min)/(n - 1) in
 * DEVICE memory, ALWAYS doubles, owned by the caller and kept alive while the context uses them.  p is interpolated
 * linearly in e (the first and last segments are continued beyond the table), c_s^2 = dp/de is the segment's slope;
 * conserved -> primitive solves E - M^2/(E + p(e)) - e = 0 by Newton's iteration, the characteristic speeds use the
 * state's own c_s^2.  Selects option "eos" = 2 ("eos" = 0 / 1 switches back; "eos" = 2 re-selects the table).
 * EINVAL: null or non-device pointer, n < 2, e_max <= e_min, or a table on another GPU than the bound workspace
 * (checked here if the workspace is bound already, else by hydro_bind_workspace). */
int hydro_set_eos_table(hydro_ctx *ctx, const void *p_device, int n, double e_min, double e_max);

/* Event-by-event batches ("event-by-event simulations"): advance nctx independent
 * contexts by nsteps CFL steps each.  The steps are issued round-robin over the batch, every context on its own
 * stream (hydro_set_stream), so that the kernels of small grids run side by side on the GPU.  Asynchronous; the
 * first error of any context is returned (its text is that context's hydro_last_error). */
int hydro_step_cfl_batch(hydro_ctx **ctxs, int nctx, double cfl, int nsteps);

/* max over interior cells and active axes of the characteristic speed a_d (a3-a4).
 * Writes one double to a HOST pointer; synchronises the stream. */
int hydro_max_signal_speed(hydro_ctx *ctx, double *out_host);

/* The same maximum for callers that cannot give the library any device memory.  Every other compute call works in the
 * workspace of hydro_bind_workspace, which somebody had to allocate.  That is not always possible: a time-step or
 * monitoring hook called from inside another code's event loop with a state it does not own; a process in which a
 * framework's memory pool holds all of the device memory and is at its cap; a latency-bound loop where cudaMalloc is
 * ruled out because it synchronises the whole device (every other event's stream would stall).  This call needs NO
 * workspace (the context may be unbound; only its grid size, "precision", equation-of-state options and stream are
 * used) and calls no cudaMalloc, cudaFree or other allocating routine: the reduction's scratch is an array built into
 * the library image, 512.25 KiB, which every GPU that loads the library holds until the process exits.
 *   cons_device          the INTERIOR state [5][nz][ny][nx] in device memory, element type per "precision" (read only)
 *   maxspeed_device_out  ONE double in device memory on the same GPU; written asynchronously on the context's stream
 *                        (a grid with no active axis gives 0)
 * Limit: the array holds one double per tile of 64 x 4 x 1 cells, at most 65536 tiles, i.e.
 * ceil(nx/64) * ceil(ny/4) * nz <= 65536 (256^3 is the largest cube).  Larger grids are refused with EINVAL and a text
 * that says so; they need hydro_max_signal_speed and a workspace.
 * Sharing: there is ONE such array per GPU and every call uses it.  Calls on the same GPU must therefore not overlap
 * in time on the device: issue them on one stream, or order the streams with events; two calls in flight at once
 * race on the array and both results are undefined.  Nothing the array held before a call is used: each call
 * zeroes the ticket counter on the stream before its kernel and overwrites the tile values it reads.
 * First call on a GPU: looks the array's device address up (cudaGetSymbolAddress, once per GPU, which also makes the
 * runtime load the library's kernels there).  Make that first call during set-up, outside any stream capture.
 * Clamped (unphysical) cells enter with their clamped speed; this call raises no flag (it has no control block).
 * EINVAL: null pointer, grid beyond the limit, pointers that are not device memory of one GPU.  ECUDA: a runtime call
 * or the launch failed.  (a3-a4 of DESIGN.md section 2; reading Q10.) */
int hydro_max_signal_speed_static(hydro_ctx *ctx, const void *cons_device, void *maxspeed_device_out);

/* L(u) of Eq. (2) for a caller-supplied interior state (DEVICE pointers, same layout as the state)
 * with ghosts filled at time t_stage: one Runge-Kutta stage's spatial operator, for per-stage parity.
 * Uses the RK stage buffers as scratch; the context's own state u^n is left untouched. */
int hydro_eval_L(hydro_ctx *ctx, const void *cons_device, double t_stage, void *L_device_out);

/* Current time (host pointer) and sticky status: HYDRO_OK or HYDRO_EUNPHYSICAL.  Both synchronise. */
int hydro_get_time(hydro_ctx *ctx, double *t_host);
int hydro_status(hydro_ctx *ctx);

/* Number of kernels the context has launched since creation (bench.py "gpu_launches"). */
long long hydro_launch_count(const hydro_ctx *ctx);

/* Slab decomposition along z: with "bc_z" = HYDRO_BC_EXTERNAL the z-ghost planes of a
 * stage input are the caller's business.  `buffer` is the state buffer that is the input of stage 0, 1, 2 of a
 * step (0 = u^n).  hydro_get_zhalo packs the g outermost INTERIOR planes of `side` (0 low z, 1 high z) into a
 * DEVICE buffer [5][g][ny][nx] (hydro_zhalo_elems elements of the context's precision); hydro_put_zhalo writes
 * such a buffer into the g GHOST planes of `side`.  hydro_step_stage runs ONE stage (0, 1, 2, in this order)
 * of a step of size dt: x/y ghost fill, the stage kernels; stage 2 also advances the time.  A driver advances
 * a slab as: for s in 0..2 { get both halos of buffer s, exchange with the neighbours, put, step_stage(dt, s) }.
 * All asynchronous on the stream.  The analytic ghost fill is not carried by the decomposition: with bc_z =
 * HYDRO_BC_EXTERNAL and HYDRO_BC_HUBBLE on x or y every stepping call returns EINVAL (the closed form needs all
 * Hubble axes and the slab's position along z). */
size_t hydro_zhalo_elems(const hydro_ctx *ctx);
int hydro_get_zhalo(hydro_ctx *ctx, int buffer, int side, void *packed_device_out);
int hydro_put_zhalo(hydro_ctx *ctx, int buffer, int side, const void *packed_device_in);
int hydro_step_stage(hydro_ctx *ctx, double dt, int stage);

/* The same without a host round trip (reading Q10 on the decomposed grid):
 *  - hydro_put_zhalo with packed_device_in == NULL fills the g ghost planes of `side` with copies of the slab's own
 *    boundary plane: the zero-gradient outflow rule (reading Q9) for a slab at a physical end of the z axis;
 *  - hydro_local_max_speed writes the max signal speed (a3-a4) of this slab's current state as ONE double to a
 *    DEVICE pointer, asynchronously (the value the last step's epilogue left, or a reduction pass); the caller
 *    max-reduces it over the slabs (ncclAllReduce on that buffer);
 *  - hydro_step_stage_cfl is hydro_step_stage with dt = cfl * dx / *maxspeed_device taken on the device in
 *    stage 0 (stages 1, 2 reuse it); maxspeed_device is a DEVICE pointer to one double and is only read.
 * EINVAL on a null pointer, cfl <= 0, or a stage out of order. */
int hydro_local_max_speed(hydro_ctx *ctx, void *maxspeed_device_out);
int hydro_step_stage_cfl(hydro_ctx *ctx, double cfl, int stage, const void *maxspeed_device);

/* One stage with the halo exchange hidden behind the interior ("fully hidden by computing the boundary
 * planes first" -- here the INTERIOR planes first, while the planes travel).  On the context's stream: x/y ghost fill,
 * the x/z kernel over the planes whose z stencils stay inside the slab, cudaStreamWaitEvent(ready_event) (a
 * cudaEvent_t the caller records on its communication stream once the neighbours' planes have arrived; NULL: no
 * wait), the ghost planes written from the packed DEVICE buffers ghosts_lo / ghosts_hi (layout of hydro_get_zhalo;
 * NULL: zero-gradient copies of the slab's own boundary plane), the x/z kernel over the g..8 outermost planes on
 * each side, the y sweep.  Results are bit-identical to hydro_put_zhalo x 2 + hydro_step_stage_cfl.  The packed
 * buffers must stay untouched until the stream has passed this call.  EINVAL unless bc_z = HYDRO_BC_EXTERNAL. */
int hydro_step_stage_overlap(hydro_ctx *ctx, double cfl, int stage, const void *maxspeed_device,
                             const void *ghosts_lo_device, const void *ghosts_hi_device, void *ready_event);

/* With the "profile" option on: total device time in milliseconds of the stage kernels (the L(u) +
 * Runge-Kutta kernel, the dominant one) launched since the last call, and their number, written to HOST
 * pointers.  Synchronises the stream and clears the record. */
int hydro_stage_kernel_time(hydro_ctx *ctx, double *ms_total_host, long long *launches_host);

/* Text of the last error on this context ("" if none).  Valid until the next call on the context. */
const char *hydro_last_error(const hydro_ctx *ctx);

void hydro_destroy(hydro_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* HYDRO_B200_H */
