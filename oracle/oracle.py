"""ctypes binding of the CPU oracle (oracle/hydro_oracle.cpp).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It does not import the CUDA package and the CUDA package does not import it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hydro_oracle.cpp")
# ORACLE_SANITIZE=1: build and load a second library compiled with -fsanitize=address,undefined (SURVEY section 5,
# sanitizers row).  The Python process must then preload the runtimes, e.g.
#   LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)" ASAN_OPTIONS=detect_leaks=0 \
#   UBSAN_OPTIONS=halt_on_error=1 ORACLE_SANITIZE=1 python -m pytest tests -m "not gpu" -q
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
_LIB = os.path.join(_HERE, "liboracle_hydro_san.so" if _SANITIZE else "liboracle_hydro.so")

OK, EINVAL, EUNPHYSICAL = 0, -1, -4


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no FMA contraction, -O2).  Returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g"] \
            if _SANITIZE else []
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-ffp-contract=off"] + san +
                              [_SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, dbl, i32 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int
        pd = ctypes.POINTER(ctypes.c_double)
        L.oracle_create.argtypes = [ctypes.POINTER(vp), i32, i32, i32, dbl, i32]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_destroy.restype = None
        L.oracle_set_option.argtypes = [vp, ctypes.c_char_p, dbl]
        L.oracle_set_state.argtypes = [vp, vp]
        L.oracle_get_state.argtypes = [vp, vp]
        L.oracle_step.argtypes = [vp, dbl, i32]
        L.oracle_max_signal_speed.argtypes = [vp, pd]
        L.oracle_get_time.argtypes = [vp, pd]
        L.oracle_eval_L.argtypes = [vp, vp, dbl, vp]
        L.oracle_eval_L_extended.argtypes = [vp, vp, dbl, vp]
        L.oracle_set_eos_table.argtypes = [vp, pd, i32, dbl, dbl]
        L.oracle_con2prim_table.argtypes = [pd, pd, i32, dbl, dbl, pd, pd]
        L.oracle_con2prim.argtypes = [pd, pd]
        L.oracle_signal_speed.argtypes = [pd, i32]
        L.oracle_signal_speed.restype = dbl
        L.oracle_phys_flux.argtypes = [pd, i32, pd]
        L.oracle_phys_flux.restype = None
        L.oracle_weno5.argtypes = [pd, dbl]
        L.oracle_weno5.restype = dbl
        L.oracle_weno7.argtypes = [pd, dbl]
        L.oracle_weno7.restype = dbl
        L.oracle_minmod.argtypes = [dbl, dbl]
        L.oracle_minmod.restype = dbl
        L.oracle_con2prim_eos.argtypes = [pd, i32, dbl, pd]
        L.oracle_signal_speed_eos.argtypes = [pd, i32, i32, dbl]
        L.oracle_signal_speed_eos.restype = dbl
        L.oracle_limited_slope.argtypes = [i32, dbl, dbl]
        L.oracle_limited_slope.restype = dbl
        L.oracle_musta_force_flux_lim.argtypes = [pd, i32, i32, dbl, i32, pd]
        L.oracle_llf_weno_flux.argtypes = [i32, pd, i32, dbl, pd]
        L.oracle_musta_force_flux.argtypes = [pd, i32, i32, dbl, pd]
        _lib = L
    return _lib


def _pd(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _arr(x, n=None):
    a = np.ascontiguousarray(x, dtype=np.float64)
    if n is not None:
        assert a.size == n, (a.shape, n)
    return a


# ---------------------------------------------------------------- pointwise pieces
def con2prim(u):
    """u = (E, Mx, My, Mz, R) -> (e, p, n, vx, vy, vz), flag."""
    u = _arr(u, 5)
    out = np.empty(6)
    flag = lib().oracle_con2prim(_pd(u), _pd(out))
    return out, flag


def signal_speed(v, d, eos=0, p0=0.0):
    v = _arr(v, 3)
    if eos:
        return lib().oracle_signal_speed_eos(_pd(v), d, int(eos), float(p0))
    return lib().oracle_signal_speed(_pd(v), d)


def con2prim_eos(u, eos, p0):
    """u -> (e, p, n, vx, vy, vz), flag for the equation of state `eos` (0: p = e/3, 1: p = p0)."""
    u = _arr(u, 5)
    out = np.empty(6)
    flag = lib().oracle_con2prim_eos(_pd(u), int(eos), float(p0), _pd(out))
    return out, flag


def con2prim_table(u, p, e_min, e_max):
    """(e, p, n, vx, vy, vz, cs2), (a_x, a_y, a_z), flag for the tabulated closure."""
    a = np.ascontiguousarray(p, dtype=np.float64)
    prim, sp = np.zeros(7), np.zeros(3)
    flag = lib().oracle_con2prim_table(_pd(_arr(u, 5)), _pd(a), len(a), float(e_min), float(e_max), _pd(prim), _pd(sp))
    return prim, sp, flag


def phys_flux(u, d):
    u = _arr(u, 5)
    out = np.empty(5)
    lib().oracle_phys_flux(_pd(u), d, _pd(out))
    return out


def weno5(f, eps=1e-6):
    f = _arr(f, 5)
    return lib().oracle_weno5(_pd(f), eps)


def weno7(f, eps=1e-6):
    f = _arr(f, 7)
    return lib().oracle_weno7(_pd(f), eps)


def minmod(a, b):
    return lib().oracle_minmod(a, b)


def llf_weno_flux(r, cells, d, eps=1e-6):
    cells = _arr(cells, 2 * r * 5)
    out = np.empty(5)
    lib().oracle_llf_weno_flux(r, _pd(cells), d, eps, _pd(out))
    return out


def limited_slope(lim, a, b):
    return lib().oracle_limited_slope(int(lim), a, b)


def musta_force_flux(cells, d, K=2, C=0.9, limiter=0):
    cells = _arr(cells, 20)
    out = np.empty(5)
    if limiter:
        lib().oracle_musta_force_flux_lim(_pd(cells), d, K, C, int(limiter), _pd(out))
    else:
        lib().oracle_musta_force_flux(_pd(cells), d, K, C, _pd(out))
    return out


# ---------------------------------------------------------------- grid solver
class Oracle:
    """Same calls as the CUDA binding (hydro_create ... hydro_get_state), host arrays."""

    def __init__(self, nx, ny, nz, dx, scheme, precision=0, **options):
        self._h = ctypes.c_void_p()
        rc = lib().oracle_create(ctypes.byref(self._h), nx, ny, nz, dx, scheme)
        if rc != OK:
            raise ValueError("oracle_create failed: %d" % rc)
        self.shape = (5, nz, ny, nx)
        self.dtype = np.float64
        for k, v in options.items():
            self.set_option(k, v)
        if precision:
            self.set_option("precision", precision)

    def set_option(self, key, value):
        rc = lib().oracle_set_option(self._h, key.encode(), float(value))
        if rc != OK:
            raise ValueError("oracle_set_option(%s=%r) failed: %d" % (key, value, rc))
        if key == "precision":
            self.dtype = np.float32 if int(value) == 1 else np.float64

    def set_state(self, cons):
        a = np.ascontiguousarray(cons, dtype=self.dtype)
        assert a.shape == self.shape, (a.shape, self.shape)
        lib().oracle_set_state(self._h, a.ctypes.data)

    def get_state(self):
        out = np.empty(self.shape, dtype=self.dtype)
        lib().oracle_get_state(self._h, out.ctypes.data)
        return out

    def step(self, dt, nsteps=1):
        return lib().oracle_step(self._h, float(dt), int(nsteps))

    def max_signal_speed(self):
        v = ctypes.c_double()
        lib().oracle_max_signal_speed(self._h, ctypes.byref(v))
        return v.value

    @property
    def time(self):
        v = ctypes.c_double()
        lib().oracle_get_time(self._h, ctypes.byref(v))
        return v.value

    def eval_L(self, cons, t_stage=0.0):
        a = np.ascontiguousarray(cons, dtype=self.dtype)
        assert a.shape == self.shape
        out = np.empty(self.shape, dtype=self.dtype)
        lib().oracle_eval_L(self._h, a.ctypes.data, float(t_stage), out.ctypes.data)
        return out

    def set_eos_table(self, p, e_min, e_max):
        """Tabulated closure p(e): values on the uniform grid e_min .. e_max; selects eos kind 2."""
        a = np.ascontiguousarray(p, dtype=np.float64)
        rc = lib().oracle_set_eos_table(self._h, _pd(a), len(a), float(e_min), float(e_max))
        assert rc == 0

    def eval_L_extended(self, cons, t_stage=0.0):
        """L(u) by the same code in long double, rounded to double (a referee for the fp64 oracle's own rounding)."""
        assert self.dtype == np.float64
        a = np.ascontiguousarray(cons, dtype=np.float64)
        assert a.shape == self.shape
        out = np.empty(self.shape, dtype=np.float64)
        rc = lib().oracle_eval_L_extended(self._h, a.ctypes.data, float(t_stage), out.ctypes.data)
        assert rc == 0
        return out

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def from_workload(w, precision=0):
    """Build an Oracle configured for a paper_1604_03360_b200.workloads.Workload (duck-typed)."""
    o = Oracle(w.n[0], w.n[1], w.n[2], w.dx, w.scheme)
    for ax, b in zip("xyz", w.bc):
        o.set_option("bc_" + ax, b)
    for ax, x0 in zip("xyz", w.origin):
        o.set_option(ax + "0", x0)
    o.set_option("t", w.t0)
    for k, v in w.options.items():
        o.set_option(k, v)
    if getattr(w, "eos_table", None) is not None:
        o.set_eos_table(*w.eos_table)
    if precision:
        o.set_option("precision", precision)
    o.set_state(w.cons)
    return o


def run(o, w, nsteps=None, dt_log=None):
    """Advance by the workload's stepping rule (Q10): fixed dt, or dt = cfl*dx/max speed per step.
    Returns the list of dt used (feed it to the other implementation for parity runs)."""
    dts = []
    for s in range(w.nsteps if nsteps is None else nsteps):
        if dt_log is not None:
            dt = dt_log[s]
        elif w.dt is not None:
            dt = w.dt
        else:
            dt = w.cfl * w.dx / o.max_signal_speed()
        o.step(dt, 1)
        dts.append(dt)
    return dts
