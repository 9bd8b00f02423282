"""Thin ctypes binding of libhydro_b200.so (include/hydro.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device memory
(the workspace and the state tensors) and for the stream handle.  Importing this module loads the
shared library and fails loudly if it has not been built; there is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os

import torch

WENO5, WENO7, MUSTA_FORCE = 0, 1, 2
BC_OUTFLOW, BC_PERIODIC, BC_HUBBLE, BC_EXTERNAL = 0, 1, 2, 3
F64, F32 = 0, 1
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_FUSED = 0, 1, 2
OK, EINVAL, ENOMEM, ECUDA, EUNPHYSICAL = 0, -1, -2, -3, -4

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhydro_b200.so")

SYMBOLS = [
    "hydro_create", "hydro_set_option", "hydro_set_stream", "hydro_workspace_bytes", "hydro_bind_workspace",
    "hydro_set_state", "hydro_get_state", "hydro_set_state_host", "hydro_get_state_host", "hydro_step",
    "hydro_step_cfl", "hydro_step_cfl_batch", "hydro_set_eos_table", "hydro_max_signal_speed",
    "hydro_max_signal_speed_static", "hydro_eval_L", "hydro_get_time", "hydro_status",
    "hydro_launch_count", "hydro_stage_kernel_time", "hydro_last_error",
    "hydro_zhalo_elems", "hydro_get_zhalo", "hydro_put_zhalo", "hydro_step_stage", "hydro_local_max_speed",
    "hydro_step_stage_cfl", "hydro_step_stage_overlap", "hydro_destroy",
]


class HydroError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("hydro error %d: %s" % (code, msg))
        self.code = code


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError("libhydro_b200.so is not built (run `python -m paper_1604_03360_b200.build`); "
                          "the hot path has no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, dbl, i32, sz = ctypes.c_void_p, ctypes.c_double, ctypes.c_int, ctypes.c_size_t
    pd = ctypes.POINTER(ctypes.c_double)
    L.hydro_create.argtypes = [ctypes.POINTER(vp), i32, i32, i32, dbl, i32]
    L.hydro_set_option.argtypes = [vp, ctypes.c_char_p, dbl]
    L.hydro_set_stream.argtypes = [vp, vp]
    L.hydro_workspace_bytes.argtypes = [vp]
    L.hydro_workspace_bytes.restype = sz
    L.hydro_bind_workspace.argtypes = [vp, vp, sz]
    L.hydro_set_state.argtypes = [vp, vp]
    L.hydro_get_state.argtypes = [vp, vp]
    L.hydro_set_state_host.argtypes = [vp, vp]
    L.hydro_get_state_host.argtypes = [vp, vp]
    L.hydro_step.argtypes = [vp, dbl, i32]
    L.hydro_step_cfl.argtypes = [vp, dbl, i32]
    L.hydro_step_cfl_batch.argtypes = [ctypes.POINTER(vp), i32, dbl, i32]
    L.hydro_set_eos_table.argtypes = [vp, vp, i32, dbl, dbl]
    L.hydro_max_signal_speed.argtypes = [vp, pd]
    L.hydro_max_signal_speed_static.argtypes = [vp, vp, vp]
    L.hydro_eval_L.argtypes = [vp, vp, dbl, vp]
    L.hydro_get_time.argtypes = [vp, pd]
    L.hydro_status.argtypes = [vp]
    L.hydro_launch_count.argtypes = [vp]
    L.hydro_launch_count.restype = ctypes.c_longlong
    L.hydro_stage_kernel_time.argtypes = [vp, pd, ctypes.POINTER(ctypes.c_longlong)]
    L.hydro_zhalo_elems.argtypes = [vp]
    L.hydro_zhalo_elems.restype = sz
    L.hydro_get_zhalo.argtypes = [vp, i32, i32, vp]
    L.hydro_put_zhalo.argtypes = [vp, i32, i32, vp]
    L.hydro_step_stage.argtypes = [vp, dbl, i32]
    L.hydro_local_max_speed.argtypes = [vp, vp]
    L.hydro_step_stage_cfl.argtypes = [vp, dbl, i32, vp]
    L.hydro_step_stage_overlap.argtypes = [vp, dbl, i32, vp, vp, vp, vp]
    L.hydro_last_error.argtypes = [vp]
    L.hydro_last_error.restype = ctypes.c_char_p
    L.hydro_destroy.argtypes = [vp]
    L.hydro_destroy.restype = None
    return L


lib = _load()


class Hydro:
    """hydro_create ... hydro_destroy with the same names; tensors in, tensors out."""

    def __init__(self, nx, ny, nz, dx, scheme, precision=F64, device="cuda", **options):
        self._h = ctypes.c_void_p()
        rc = lib.hydro_create(ctypes.byref(self._h), nx, ny, nz, float(dx), scheme)
        if rc != OK:
            raise HydroError(rc, "hydro_create(%d,%d,%d,%g,%d)" % (nx, ny, nz, dx, scheme))
        self.shape = (5, nz, ny, nx)
        self.device = torch.device(device)
        self.dtype = torch.float32 if precision == F32 else torch.float64
        self._ws = None
        if precision != F64:
            self.set_option("precision", precision)
        for k, v in options.items():
            self.set_option(k, v)

    def _check(self, rc):
        if rc != OK:
            raise HydroError(rc, lib.hydro_last_error(self._h).decode())

    def set_option(self, key, value):
        self._check(lib.hydro_set_option(self._h, key.encode(), float(value)))

    def set_eos_table(self, p, e_min, e_max):
        """Tabulated closure p(e): `p` = values on the uniform grid e_min .. e_max (any array-like; uploaded as a
        float64 device tensor that this object keeps alive)."""
        self._eos_table = torch.as_tensor(p, dtype=torch.float64).to(self.device).contiguous()
        self._check(lib.hydro_set_eos_table(self._h, self._eos_table.data_ptr(), self._eos_table.numel(),
                                            float(e_min), float(e_max)))

    def workspace_bytes(self):
        return lib.hydro_workspace_bytes(self._h)

    def bind(self):
        """Allocate the workspace with torch and hand it to the library; use torch's current stream."""
        nbytes = self.workspace_bytes()
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self._ws.data_ptr() + 255) // 256 * 256
        self._check(lib.hydro_set_stream(self._h, torch.cuda.current_stream(self.device).cuda_stream))
        self._check(lib.hydro_bind_workspace(self._h, ptr, nbytes))
        return self

    def set_stream(self, stream):
        self._check(lib.hydro_set_stream(self._h, stream.cuda_stream))

    def _dev(self, t):
        assert t.is_cuda and t.is_contiguous() and t.dtype == self.dtype and tuple(t.shape) == self.shape, \
            (t.device, t.dtype, tuple(t.shape), self.shape)
        return t.data_ptr()

    def _host(self, t):
        assert (not t.is_cuda) and t.is_contiguous() and t.dtype == self.dtype and tuple(t.shape) == self.shape
        return t.data_ptr()

    def set_state(self, cons):
        self._check(lib.hydro_set_state(self._h, self._dev(cons)))

    def get_state(self, out=None):
        if out is None:
            out = torch.empty(self.shape, dtype=self.dtype, device=self.device)
        self._check(lib.hydro_get_state(self._h, self._dev(out)))
        return out

    def set_state_host(self, cons_host):
        self._check(lib.hydro_set_state_host(self._h, self._host(cons_host)))

    def get_state_host(self, out_host):
        self._check(lib.hydro_get_state_host(self._h, self._host(out_host)))
        return out_host

    def step(self, dt, nsteps=1):
        self._check(lib.hydro_step(self._h, float(dt), int(nsteps)))

    def step_cfl(self, cfl, nsteps=1):
        self._check(lib.hydro_step_cfl(self._h, float(cfl), int(nsteps)))

    def max_signal_speed(self):
        v = ctypes.c_double()
        self._check(lib.hydro_max_signal_speed(self._h, ctypes.byref(v)))
        return v.value

    def max_signal_speed_static(self, cons, out):
        """hydro_max_signal_speed_static: max signal speed of the interior state `cons` into the 1-element float64
        device tensor `out`, asynchronously, with no workspace (the context need not be bound) and no allocation here
        or in the library: for callers that cannot allocate device memory (see include/hydro.h).  Grids up to
        ceil(nx/64) * ceil(ny/4) * nz = 65536 tiles; calls on one GPU must not overlap."""
        assert out.is_cuda and out.dtype == torch.float64 and out.numel() == 1 and out.device == cons.device
        self._check(lib.hydro_max_signal_speed_static(self._h, self._dev(cons), out.data_ptr()))
        return out

    def eval_L(self, cons, t_stage=0.0, out=None):
        if out is None:
            out = torch.empty(self.shape, dtype=self.dtype, device=self.device)
        self._check(lib.hydro_eval_L(self._h, self._dev(cons), float(t_stage), self._dev(out)))
        return out

    @property
    def time(self):
        v = ctypes.c_double()
        self._check(lib.hydro_get_time(self._h, ctypes.byref(v)))
        return v.value

    def status(self):
        return lib.hydro_status(self._h)

    @property
    def launch_count(self):
        return lib.hydro_launch_count(self._h)

    def zhalo_elems(self):
        return lib.hydro_zhalo_elems(self._h)

    def get_zhalo(self, buffer, side, out=None):
        if out is None:
            out = torch.empty(self.zhalo_elems(), dtype=self.dtype, device=self.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == self.dtype and out.numel() == self.zhalo_elems()
        self._check(lib.hydro_get_zhalo(self._h, int(buffer), int(side), out.data_ptr()))
        return out

    def put_zhalo(self, buffer, side, packed):
        """packed = None: zero-gradient ghosts from the slab's own boundary plane (a physical outflow end)."""
        if packed is None:
            self._check(lib.hydro_put_zhalo(self._h, int(buffer), int(side), None))
            return
        assert packed.is_cuda and packed.is_contiguous() and packed.dtype == self.dtype and packed.numel() == self.zhalo_elems()
        self._check(lib.hydro_put_zhalo(self._h, int(buffer), int(side), packed.data_ptr()))

    def local_max_speed(self, out=None):
        """Max signal speed of this context's state as a 1-element float64 DEVICE tensor (no host sync)."""
        if out is None:
            out = torch.empty(1, dtype=torch.float64, device=self.device)
        assert out.is_cuda and out.dtype == torch.float64 and out.numel() == 1
        self._check(lib.hydro_local_max_speed(self._h, out.data_ptr()))
        return out

    def step_stage_cfl(self, cfl, stage, maxspeed):
        assert maxspeed.is_cuda and maxspeed.dtype == torch.float64 and maxspeed.numel() == 1
        self._check(lib.hydro_step_stage_cfl(self._h, float(cfl), int(stage), maxspeed.data_ptr()))

    def step_stage(self, dt, stage):
        self._check(lib.hydro_step_stage(self._h, float(dt), int(stage)))

    def step_stage_overlap(self, cfl, stage, maxspeed, ghosts_lo, ghosts_hi, ready_event=None):
        """hydro_step_stage_overlap; ghosts_* = packed device tensors or None (zero-gradient); ready_event = a
        torch.cuda.Event recorded on the communication stream, or None."""
        assert maxspeed.is_cuda and maxspeed.dtype == torch.float64 and maxspeed.numel() == 1
        for t in (ghosts_lo, ghosts_hi):
            assert t is None or (t.is_cuda and t.is_contiguous() and t.dtype == self.dtype and t.numel() == self.zhalo_elems())
        ev = None if ready_event is None else ctypes.c_void_p(ready_event.cuda_event)
        self._check(lib.hydro_step_stage_overlap(self._h, float(cfl), int(stage), maxspeed.data_ptr(),
                                                 None if ghosts_lo is None else ghosts_lo.data_ptr(),
                                                 None if ghosts_hi is None else ghosts_hi.data_ptr(), ev))

    def stage_kernel_time(self):
        """(total ms, launches) of the stage kernels since the last call ("profile" option)."""
        ms, n = ctypes.c_double(), ctypes.c_longlong()
        self._check(lib.hydro_stage_kernel_time(self._h, ctypes.byref(ms), ctypes.byref(n)))
        return ms.value, n.value

    def close(self):
        if getattr(self, "_h", None):
            lib.hydro_destroy(self._h)
            self._h = ctypes.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def step_cfl_batch(hydros, cfl, nsteps=1):
    """hydro_step_cfl_batch: advance independent contexts (each bound to its own stream) round-robin."""
    arr = (ctypes.c_void_p * len(hydros))(*[h._h for h in hydros])
    rc = lib.hydro_step_cfl_batch(arr, len(hydros), float(cfl), int(nsteps))
    if rc != OK:
        for h in hydros:
            msg = lib.hydro_last_error(h._h).decode()
            if msg:
                raise HydroError(rc, msg)
        raise HydroError(rc, "hydro_step_cfl_batch")


def from_workload(w, precision=F64, kernel=KERNEL_AUTO, device="cuda"):
    """Context configured for a workloads.Workload, state uploaded (host numpy -> device)."""
    h = Hydro(w.n[0], w.n[1], w.n[2], w.dx, w.scheme, precision=precision, device=device)
    for ax, b in zip("xyz", w.bc):
        h.set_option("bc_" + ax, b)
    for ax, x0 in zip("xyz", w.origin):
        h.set_option(ax + "0", x0)
    h.set_option("t", w.t0)
    h.set_option("kernel", kernel)
    for k, v in w.options.items():
        h.set_option(k, v)
    if getattr(w, "eos_table", None) is not None:
        h.set_eos_table(*w.eos_table)
    h.bind()
    h.set_state(torch.from_numpy(w.cons).to(device=device, dtype=h.dtype).contiguous())
    return h
