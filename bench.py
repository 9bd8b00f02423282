#!/usr/bin/env python
"""bench.py -- throughput of the hot path (three L(u) + SSP-RK3 combine per step) on
BASELINE.json configs[4]: the 512^3 periodic lumpy state with 200 hotspots and blended velocities.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--scheme weno5|weno7|musta] [--precision f64|f32]
                    [--grid 512] [--no-variants] [--no-cpu-baseline] [--impl reference]

One "step" is one SSP-RK3 step of the whole grid with dt = CFL dx / max signal speed taken on the device
(hydro_step_cfl, reading Q10): per stage the ghost fill, the x/z marching kernel and the y sweep; both make con2prim
and the signal speeds of the cells they read on the fly, and the stage-3 y sweep's epilogue reduces the CFL maximum
of the new state for the next step.
Prints ONE JSON line (rank 0).  N > 1 (torchrun): ONE 512^3 event decomposed into z-slabs with a halo exchange per
Runge-Kutta stage (`--decomp slab`, the default for N > 1: SURVEY 8(e), strong scaling), time = max over ranks; the
throughput of N independent events (`--decomp events`, weak scaling, no data-path collective) is printed beside it
as `replicas`.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same
workload on the host cores; it is the only other place besides `cpu_baseline` where bench.py runs it.
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1604_03360_b200 import workloads as W  # noqa: E402

SCHEMES = {"weno5": W.WENO5, "weno7": W.WENO7, "musta": W.MUSTA_FORCE}
# Algorithmic flops per cell per RK3 step and bytes per cell per RK3 step (
# SURVEY.md 8(d)): add/mul/div/sqrt/max = 1, FMA = 2, every interface flux computed once.
FLOPS_PER_CELL_STEP = {"weno5": 7041.0, "weno7": 14331.0, "musta": 3831.0}
FLOPS_PER_CELL_L = {"weno5": 2327.0, "weno7": 4757.0, "musta": 1257.0}
BYTES_PER_CELL_STEP = {"f64": 320.0, "f32": 160.0}
# DRAM bytes of one stage (x/z kernel + y sweep) = dram__bytes_read.sum + dram__bytes_write.sum of both launches, per
# scheme and per Runge-Kutta stage, from the ncu pass over a whole step of each scheme at 512^3
# (profiles/r03_traffic.md, raw lists profiles/r03_traffic_<scheme>.csv).  Stage 1 does not read u^n; stages 2 and 3
# do (+5.4e9).  Algorithmic bytes per stage at that size: 80 / 120 / 120 B x 512^3 = 1.07e10 / 1.61e10 / 1.61e10.
TRAFFIC_BYTES_PER_STAGE = {("weno5", "f64", 512): (27.59e9, 33.10e9, 32.97e9),
                           ("weno7", "f64", 512): (27.59e9, 33.09e9, 33.05e9),
                           ("musta", "f64", 512): (27.61e9, 33.06e9, 32.92e9)}
KERNEL_NAMES = {"weno5": "weno_xz_kernel<T,3> + weno_y_kernel<T,3,EPI>", "weno7": "weno_xz_kernel<T,4> + weno_y_kernel<T,4,EPI>",
                "musta": "musta_xz_kernel<T,FAST> + musta_y_kernel<T,EPI,FAST>"}
METRIC = "3D cell-updates/s per RK3 step"
UNIT = "cell-updates/s"
CFL = 0.2


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, power, reasons = [], None, [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for t, line in self.rows:
            if not (t0 <= t <= t1 + 0.1):
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0]))
                smax = float(f[1])
                power.append(float(f[2]))
            except Exception:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        hist = {}
        for v in sm:                                   # SM clock histogram in 50 MHz bins (lower edge -> samples)
            b = str(int(v // 50 * 50))
            hist[b] = hist.get(b, 0) + 1
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "power_w": float(np.median(power)) if power else None,
                "power_w_max": max(power) if power else None, "sm_mhz_hist": hist,
                "samples": len(sm), "reasons": sorted(reasons)}


def make_workload(n, scheme, rank=0):
    if n >= 64:
        w = W.lumpy(n=n, hotspots=200, with_velocity=True, scheme=SCHEMES[scheme], nsteps=20, cfl=CFL,
                    seed=W.SEED + rank)
    else:
        w = W.lumpy(n=n, hotspots=12, with_velocity=True, scheme=SCHEMES[scheme], box=n / 16.0, sigma_unit=0.12)
    return w


CPU_CROP = 48


def oracle_sample(n, scheme, m=CPU_CROP):
    """The oracle's bounded sample of the bench workload: the corner block of the first m cells per axis of the
    same seeded n^3 state (same draws and formulas as make_workload(n, scheme), evaluated on those cells only),
    made periodic by fiat."""
    if n >= 64:
        return W.lumpy(n=n, hotspots=200, with_velocity=True, scheme=SCHEMES[scheme], nsteps=20, cfl=CFL,
                       crop=min(m, n))
    w = make_workload(n, scheme)
    return W.Workload(w.name + "_crop", w.n, w.dx, (0.0, 0.0, 0.0), w.scheme, w.bc, w.cons, 0.0, cfl=w.cfl,
                      nsteps=w.nsteps)


def time_oracle(w, steps, warmup=0):
    """Cell-updates/s of the oracle as it stands, single-threaded, on workload w."""
    from oracle import oracle as O
    o = O.from_workload(w)
    for _ in range(warmup):
        o.step(w.cfl * w.dx / o.max_signal_speed(), 1)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(w.cfl * w.dx / o.max_signal_speed(), 1)
    dt = time.perf_counter() - t0
    ncell = w.n[0] * w.n[1] * w.n[2]
    o.close()
    return ncell * steps / dt, dt


def oracle_all_cores(n, scheme, steps, timeout=240):
    """one independent single-threaded oracle process per host core (`bench.py --oracle-worker`),
    each on the same sample; aggregate = all cell-updates done / the slowest process's time."""
    try:
        cores = len(os.sched_getaffinity(0))
    except AttributeError:
        cores = os.cpu_count() or 1
    env = dict(os.environ, OMP_NUM_THREADS="1", OPENBLAS_NUM_THREADS="1", MKL_NUM_THREADS="1")
    cmd = [sys.executable, os.path.abspath(__file__), "--oracle-worker", "--grid", str(n), "--scheme", scheme,
           "--steps", str(steps)]
    procs = [subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True, env=env)
             for _ in range(cores)]
    res = []
    deadline = time.time() + timeout
    for p in procs:
        try:
            out, _ = p.communicate(timeout=max(1.0, deadline - time.time()))
            ncell, secs = out.strip().split()[-2:]
            res.append((int(ncell), float(secs)))
        except Exception:
            p.kill()
    if not res:
        return None, None, 0
    slowest = max(r[1] for r in res)
    return len(res) * res[0][0] * steps / slowest, slowest, len(res)


def oracle_worker(args):
    """One process of the all-core leg: prints `ncell seconds`."""
    w = oracle_sample(args.n, args.scheme)
    _, secs = time_oracle(w, args.steps)
    print(w.n[0] * w.n[1] * w.n[2], secs, flush=True)
    return 0


def cpu_baseline(n, scheme, steps):
    w = oracle_sample(n, scheme)
    m = w.n[0]
    v1, s1 = time_oracle(w, steps)
    vall, sall, cores = oracle_all_cores(n, scheme, steps)
    return {"value": vall, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d^3 corner block of the same %d^3 state, %d RK3 steps: one independent single-threaded oracle "
                      "process per host core (%d cores, %.1f s); host has %d logical CPUs" %
                      (m, n, steps, cores, sall, os.cpu_count() or 0),
            "single_thread": {"value": v1, "cores": 1, "seconds": s1}}


# ----------------------------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = oracle_sample(args.n, args.scheme)
    m = w.n[0]
    value, secs = time_oracle(w, args.steps, args.warmup)
    sample = ("%d^3 corner block of the same seeded %d^3 state the GPU arm advances, %d RK3 steps after %d warm-up, "
              "1 thread" % (m, args.n, args.steps, args.warmup))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[4]: %d^3 periodic lumpy state, 200 hotspots, blended velocities, "
                               "%s f64, CFL %.1f; the oracle (oracle/, as it stands) on a bounded sample: %s" %
                               (args.n, args.scheme, CFL, sample),
                   "grid": [args.n] * 3, "scheme": args.scheme, "cfl": CFL, "sample_grid": [m] * 3},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def probe_fma_peak(torch, precision, millis=300):
    """Sustained FMA rate in TFLOP/s from the bench-side helper library (csrc/bench_probe.cu); None if it is absent."""
    path = os.path.join(ROOT, "paper_1604_03360_b200", "libbench_probe.so")
    if not os.path.exists(path):
        return None
    lib = ctypes.CDLL(path)
    lib.bench_probe_fma_peak.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                         ctypes.POINTER(ctypes.c_double)]
    scratch = torch.zeros(16, dtype=torch.uint8, device="cuda")
    out = ctypes.c_double()
    rc = lib.bench_probe_fma_peak(0 if precision == "f64" else 1, millis, torch.cuda.current_stream().cuda_stream,
                                  scratch.data_ptr(), ctypes.byref(out))
    return out.value if rc == 0 else None


# ----------------------------------------------------------------------------------------------

def timed_run(B, torch, w, precision, steps, warmup, dist=None, profile=True, slab=None):
    """Warm up, then time `steps` RK3 steps with CUDA events on the stream.  Returns a dict.
    slab = (rank, world): this rank owns one z-slab of the global grid and exchanges halo planes with its
    neighbours every stage (paper_1604_03360_b200/slab.py); otherwise the rank advances the whole grid."""
    prec = B.F32 if precision == "f32" else B.F64
    if slab is None:
        h = B.from_workload(w, precision=prec)
        advance = lambda k: h.step_cfl(CFL, k)
    else:
        from paper_1604_03360_b200 import slab as S
        rank, world = slab
        k0, k1 = S.split_planes(w.n[2], world)[rank]
        h = S.make_slab(B, w, k0, k1, precision=prec)
        comm = S.DistComm(dist, w.bc[2]) if dist is not None else S.LocalComm(1, w.bc[2])
        group = S.SlabGroup([h], comm, w.dx)
        advance = lambda k: group.step_cfl(CFL, k)
    stream = torch.cuda.current_stream()
    advance(warmup)
    torch.cuda.synchronize()
    if profile:
        h.set_option("profile", 1)
    l0 = h.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0.record(stream)
    for _ in range(steps):
        advance(1)
    e1.record(stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    if dist is not None:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    launches = h.launch_count - l0
    stage_ms, stage_n = h.stage_kernel_time() if profile else (0.0, 0)
    h.set_option("profile", 0)
    status = h.status()
    tnow = h.time
    return dict(h=h, ms=ms, launches=launches, stage_ms=stage_ms, stage_n=stage_n, status=status, t=tnow,
                wall=(t0, t1), advance=advance)


def max_over_ranks(value, dist=None, device="cpu"):
    """Max of a scalar over all ranks (the multi-GPU timing rule); identity without a process group."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(ncell, steps, world, ms):
    """Whole-job cell-updates/s: every rank advances its own event of ncell cells (weak scaling)."""
    return ncell * steps * world / (ms * 1e-3)


def roofline(scheme, precision, ncell, stage_ms, stage_n, alu_peak_tf, peaks, probe_tf=None, step_ms=None):
    """Roofline object of the dominant "kernel" = one RK stage's pair of stage kernels (x/z marching kernel + y
    sweep), timed together by one CUDA-event pair per stage on the launching stream inside the timed region."""
    if stage_n == 0 or stage_ms <= 0:
        return None
    per_launch_s = stage_ms * 1e-3 / stage_n
    flops = FLOPS_PER_CELL_L[scheme] * ncell
    achieved = flops / per_launch_s / 1e12
    byts = BYTES_PER_CELL_STEP[precision] / 3.0 * ncell
    r = {"bound": "alu", "achieved": achieved, "peak": alu_peak_tf, "unit": "TFLOP/s",
         "frac": achieved / alu_peak_tf, "frac_is": "of the NOMINAL fp peak (clocks.max.sm)",
         "traffic": (lambda t: sum(t) / 3.0 if t else None)(
             TRAFFIC_BYTES_PER_STAGE.get((scheme, precision, round(ncell ** (1.0 / 3.0))))),
         "traffic_per_stage": TRAFFIC_BYTES_PER_STAGE.get((scheme, precision, round(ncell ** (1.0 / 3.0)))),
         "traffic_note": "DRAM bytes (read + write, both kernels) of one stage launch: mean over the three stages of a "
                         "step, and stage 1 / 2 / 3 beside it, from the ncu pass of this scheme under "
                         "profiles/r03_traffic.md; algorithmic bytes of a mean stage: %.3g" % byts,
         "kernel": "one RK stage = %s, timed together with one CUDA-event pair on the stream" % KERNEL_NAMES[scheme],
         "launch_ms": per_launch_s * 1e3, "algorithmic_flops_per_launch": flops,
         "hbm_gbs_achieved": byts / per_launch_s / 1e9, "hbm_frac": byts / per_launch_s / 1e9 / peaks["hbm_gbs"]}
    if probe_tf:
        r["peak_probe_sustained"] = probe_tf
        r["frac_of_probe"] = achieved / probe_tf
    if step_ms:
        r["stage_share_of_step"] = stage_ms / step_ms
    return r


def batch_bench(B, torch, scheme, n=128, nb=8, steps=10, warmup=3):
    """SURVEY 8(f)-N2 / N4 ("event-by-event simulations"): nb independent n^3 events.  (a) one after the
    other on one stream, (b) hydro_step_cfl_batch with one stream per event, (c) the same with every event's step
    replayed from a CUDA graph -- all `steps` steps of an event from ONE graph launch.  Whole-batch cell-updates/s,
    CUDA events around the batch; host_enqueue_ms_per_step = host time spent issuing the work, per step of the batch."""
    ws = [make_workload(n, scheme, rank=k) for k in range(nb)]
    out = {"grid": [n, n, n], "events": nb, "steps": steps, "unit": UNIT}
    for mode in ("sequential", "streams", "streams+graph"):
        streams = [torch.cuda.Stream() for _ in range(nb)]
        hs = []
        for w, st in zip(ws, streams):
            with torch.cuda.stream(st if mode != "sequential" else streams[0]):
                h = B.from_workload(w)
                if mode == "streams+graph":
                    h.set_option("graph", 1)
                hs.append(h)
        def advance(k):
            if mode == "sequential":
                for h in hs:
                    h.step_cfl(CFL, k)
            else:
                B.step_cfl_batch(hs, CFL, k)
        advance(warmup)
        advance(steps)            # untimed: the k-step graph of (c) is captured and instantiated on its first use
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(torch.cuda.default_stream())
        for st in streams:
            st.wait_event(e0)
        tq = time.perf_counter()
        advance(steps)
        enqueue_s = time.perf_counter() - tq
        for st in streams:
            torch.cuda.default_stream().wait_stream(st)
        e1.record(torch.cuda.default_stream())
        torch.cuda.synchronize()
        host_s = time.perf_counter() - t0
        ms = e0.elapsed_time(e1)
        out[mode] = {"value": nb * n ** 3 * steps / (ms * 1e-3), "ms_per_step_per_event": ms / steps / nb,
                     "host_seconds": host_s, "host_enqueue_ms_per_step": enqueue_s / steps * 1e3,
                     "status": max(h.status() for h in hs)}
        for h in hs:
            h.close()
        torch.cuda.empty_cache()
    return out


def nominal_tflops(sms, precision, peaks):
    lanes = 64 if precision == "f64" else 128
    return sms * lanes * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12, lanes


def run_ours(args):
    import torch
    if not torch.cuda.is_available():
        print("bench.py: no CUDA device; the hot path has no CPU fallback", file=sys.stderr)
        return 2
    from paper_1604_03360_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist = dist_mod
    peaks, peaks_src = measured_peaks()

    n = args.n
    ncell = n ** 3
    decomp = args.decomp or ("slab" if world > 1 else "events")
    slab_mode = decomp == "slab"
    # events: every rank its own event (seeded by rank); slab: ONE global event, this rank owns a z-slab of it
    w = make_workload(n, args.scheme, 0 if slab_mode else rank)
    slab = (rank, world) if slab_mode else None

    # ALU roofline denominator: 148 SMs x 64 fp64 (128 fp32) FMA lanes x 2 flop x
    # the SM clock.  Nominal uses clocks.max.sm; the sustained figure is measured by the bench-side probe.
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    nominal_tf, lanes = nominal_tflops(sms, args.precision, peaks)
    probe_tf = {p: probe_fma_peak(torch, p, 300) for p in ("f64", "f32")}

    sampler = ClockSampler(local)
    sampler.start()
    r = timed_run(B, torch, w, args.precision, args.steps, args.warmup, dist, slab=slab)
    clocks = sampler.stop(*r["wall"])
    ms = max_over_ranks(r["ms"], dist, "cuda")
    value = aggregate_value(ncell, args.steps, 1 if slab_mode else world, ms)
    ncell_local = ncell // world if slab_mode else ncell
    roof = roofline(args.scheme, args.precision, ncell_local, r["stage_ms"], r["stage_n"], nominal_tf, peaks,
                    probe_tf[args.precision], r["ms"])
    if roof is not None:
        roof["peak_source"] = ("nominal: %d SMs x %d lanes x 2 x %.0f MHz (DESIGN.md section 8); "
                               "hbm peak %s" % (sms, lanes, peaks.get("sm_max_mhz", 1965.0), peaks_src))
    # step-level roofline: cell-updates/s against min(byte roof, flop roof)
    flop_roof = nominal_tf * 1e12 / FLOPS_PER_CELL_STEP[args.scheme]
    byte_roof = peaks["hbm_gbs"] * 1e9 / BYTES_PER_CELL_STEP[args.precision]
    step_roof = min(flop_roof, byte_roof)

    h = r.pop("h")
    advance = r.pop("advance")
    stream = torch.cuda.current_stream()

    # ---- median of >= 5 repetitions of the K-step run (the first is the one `value` reports)
    reps = [ms / max(args.steps, 1)]
    for _ in range(max(0, args.repeat - 1)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        e0.record(stream)
        for _k in range(args.steps):
            advance(1)
        e1.record(stream)
        torch.cuda.synchronize()
        reps.append(max_over_ranks(e0.elapsed_time(e1), dist, "cuda") / max(args.steps, 1))
    repetitions = {"ms_per_step": reps, "median_ms_per_step": float(np.median(reps)),
                   "median_value": (ncell if slab_mode else ncell * world) / (float(np.median(reps)) * 1e-3)}

    # ---- e2e: host buffers through the C ABI, copies inside the timed region
    esz = 8 if args.precision == "f64" else 4
    tdt = torch.float64 if args.precision == "f64" else torch.float32
    if slab_mode:
        from paper_1604_03360_b200 import slab as S
        k0, k1 = S.split_planes(n, world)[rank]
        host_in = torch.from_numpy(np.ascontiguousarray(w.cons[:, k0:k1])).to(tdt)
    else:
        host_in = torch.from_numpy(w.cons).to(tdt)
    host_out = torch.empty_like(host_in)
    pinned = True
    try:
        host_in, host_out = host_in.pin_memory(), host_out.pin_memory()
    except RuntimeError:
        pinned = False                 # many ranks on one host can exhaust lockable memory: pageable copies then
    h.set_state_host(host_in)          # warm the copy path
    advance(1)
    h.get_state_host(host_out)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    h.set_state_host(host_in)
    advance(args.steps)
    h.get_state_host(host_out)
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0, dist, "cuda")
    state_bytes = 5 * ncell_local * esz
    e2e = {"value": aggregate_value(ncell, args.steps, 1 if slab_mode else world, e2e_s * 1e3), "unit": UNIT,
           "h2d_bytes_per_step": state_bytes / max(args.steps, 1),
           "d2h_bytes_per_step": state_bytes / max(args.steps, 1),
           "pinned_host_memory": pinned,
           "job": "hydro_set_state_host + %d steps + hydro_get_state_host; "
                  "state %d bytes each way per job and rank" % (args.steps, state_bytes),
           "finite": bool(torch.isfinite(host_out).all().item())}
    launches_per_step = r["launches"] / max(args.steps, 1)
    h.close()
    del h, host_in, host_out
    torch.cuda.empty_cache()

    # ---- N > 1, slab: the throughput of N independent events beside it (no data-path collective)
    replicas = None
    if slab_mode and world > 1:
        rr = timed_run(B, torch, w, args.precision, max(3, args.steps // 4), 3, dist, profile=False)
        rms = max_over_ranks(rr["ms"], dist, "cuda")
        replicas = {"value": aggregate_value(ncell, max(3, args.steps // 4), world, rms), "unit": UNIT,
                    "scaling": "weak", "note": "one independent %d^3 event per GPU, no exchange" % n,
                    "ms_per_step": rms / max(3, args.steps // 4)}
        rr.pop("h").close()
        torch.cuda.empty_cache()

    # ---- the other headline variants of config 5: full lines (same grid, same number of steps, own clocks)
    variants = {}
    if not args.no_variants and rank == 0 and world == 1 and not slab_mode:
        for sch, prec in (("weno5", "f64"), ("weno7", "f64"), ("musta", "f64"), ("weno5", "f32"), ("weno7", "f32")):
            if (sch, prec) == (args.scheme, args.precision):
                continue
            w.scheme = SCHEMES[sch]
            vs = ClockSampler(local)
            vs.start()
            vr = timed_run(B, torch, w, prec, args.steps, args.warmup)
            vclk = vs.stop(*vr["wall"])
            nom_v, _ = nominal_tflops(sms, prec, peaks)
            rf = roofline(sch, prec, ncell, vr["stage_ms"], vr["stage_n"], nom_v, peaks, probe_tf[prec], vr["ms"])
            variants["%s_%s" % (sch, prec)] = {
                "value": ncell * args.steps / (vr["ms"] * 1e-3), "ms_per_step": vr["ms"] / args.steps,
                "steps": args.steps, "warmup": args.warmup, "dtype": prec,
                "roofline_frac": rf["frac"] if rf else None, "roofline": rf,
                "step_roofline_frac": (ncell * args.steps / (vr["ms"] * 1e-3)) /
                                      min(nom_v * 1e12 / FLOPS_PER_CELL_STEP[sch],
                                          peaks["hbm_gbs"] * 1e9 / BYTES_PER_CELL_STEP[prec]),
                "launches_per_step": vr["launches"] / args.steps, "clocks": vclk, "status": vr["status"]}
            vr.pop("h").close()
            torch.cuda.empty_cache()
        w.scheme = SCHEMES[args.scheme]

    # ---- the same scheme at 128^3 and 256^3
    sizes = {}
    if not args.no_variants and rank == 0 and world == 1 and not slab_mode:
        for m in (128, 256):
            if m >= n:
                continue
            wm = make_workload(m, args.scheme)
            sr = timed_run(B, torch, wm, args.precision, args.steps, args.warmup, profile=False)
            sizes[str(m)] = {"value": m ** 3 * args.steps / (sr["ms"] * 1e-3), "ms_per_step": sr["ms"] / args.steps,
                             "steps": args.steps, "launches_per_step": sr["launches"] / args.steps}
            sr.pop("h").close()
            torch.cuda.empty_cache()

    # ---- a batch of small events on streams, with and without the CUDA-graph replay
    batch = None
    if not args.no_variants and rank == 0 and world == 1 and not slab_mode:
        batch = batch_bench(B, torch, args.scheme, n=128, nb=8, steps=args.steps)
        batch["at_64"] = batch_bench(B, torch, args.scheme, n=64, nb=8, steps=args.steps)

    # ---- the oracle beside it: bounded sample on the host cores (rank 0, N = 1 only)
    cpu = None
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        cpu = cpu_baseline(n, args.scheme, 16)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / max(args.steps, 1), "higher_is_better": True,
            "scaling": "strong" if slab_mode else "weak", "vs_baseline": None, "dtype": args.precision,
            "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[4]: %d^3 periodic lumpy state, 200 hotspots, blended "
                                   "velocities, %s %s, CFL %.1f (%s)" %
                                   (n, args.scheme, args.precision, CFL,
                                    "one event, z-slab per GPU, halo exchange per stage" if slab_mode
                                    else "one independent event per GPU"),
                       "grid": [n, n, n], "scheme": args.scheme, "cfl": CFL, "decomp": decomp,
                       "l2": "no flush needed: the state (%.2f GB per copy) is far larger than the 126 MB L2" %
                             (state_bytes / 1e9)},
            "roofline": roof,
            "step_roofline": {"value": value / world, "roof": step_roof, "frac": value / world / step_roof,
                              "per": "GPU",
                              "flop_roof": flop_roof, "byte_roof": byte_roof, "unit": UNIT,
                              "note": "min(hbm peak / 320 B, nominal ALU peak / algorithmic flops) per cell-update"},
            "repetitions": repetitions,
            "cpu_baseline": cpu,
            "e2e": e2e,
            "gpu_launches": int(round(launches_per_step * args.steps)),
            "launches_per_step": launches_per_step,
            "clocks": clocks,
            "status": r["status"], "sim_time": r["t"],
            "variants": variants,
            "sizes": sizes,
            "replicas": replicas,
            "batch": batch,
            "context": "paper: GPU ~200x one CPU thread for MUSTA-FORCE on unnamed 2016 hardware (PAPER.md:38)",
        }
        # last key, so that a record that keeps only the tail of this line still holds every variant's numbers:
        # [ms per step, stage-kernel roofline fraction of the nominal peak, median SM MHz, median W]
        summary = {"%s_%s" % (args.scheme, args.precision): [round(ms / max(args.steps, 1), 3),
                                                             round(roof["frac"], 4) if roof else None,
                                                             clocks.get("sm_mhz"), clocks.get("power_w")]}
        for k, v in variants.items():
            summary[k] = [round(v["ms_per_step"], 3), round(v["roofline_frac"], 4) if v["roofline_frac"] else None,
                          v["clocks"].get("sm_mhz"), v["clocks"].get("power_w")]
        line["variants_summary"] = summary
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scheme", default="weno5", choices=sorted(SCHEMES))
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--grid", "--n", dest="n", type=int, default=512,
                    help="cells per axis (use --grid under torchrun: its parser finds --n ambiguous)")
    ap.add_argument("--no-variants", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--repeat", type=int, default=5, help="repetitions of the K-step run for the median (first = value)")
    ap.add_argument("--decomp", default=None, choices=["events", "slab"],
                    help="'slab' (default for N > 1) = one event decomposed along z, halo exchange per stage (strong "
                         "scaling); 'events' (default for N = 1) = one independent event per GPU (weak scaling, no "
                         "data-path collective)")
    ap.add_argument("--oracle-worker", action="store_true", help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.oracle_worker:
        return oracle_worker(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
