"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle side (``oracle/``, ``tests/``) and the
CUDA side (``bench.py``, ``-m gpu`` tests).  It holds no step of the hot path: it builds primitive
fields (e, n, v) from the recipes in DESIGN.md section 4 / SURVEY.md section 8(d) and converts
them to the conserved variables by their *definition* (SURVEY.md section 8 notation,
PAPER.md:15 "energy density, momenta densities and conserved charge densities"):

    E = (e+p) gamma^2 - p,   M_i = (e+p) gamma^2 v_i,   R = n gamma,   p = e/3.

Arrays are float64, layout [5][nz][ny][nx] (x fastest), field order E, Mx, My, Mz, R.
numpy only; importing it never touches CUDA or the oracle.
"""
from __future__ import annotations

import dataclasses
import numpy as np

SEED = 1604  # numpy default_rng(1604)

WENO5, WENO7, MUSTA_FORCE = 0, 1, 2
BC_OUTFLOW, BC_PERIODIC, BC_HUBBLE = 0, 1, 2


@dataclasses.dataclass
class Workload:
    name: str
    n: tuple            # (nx, ny, nz)
    dx: float
    origin: tuple       # coordinate of the low face of the domain on each axis
    scheme: int
    bc: tuple           # per axis
    cons: np.ndarray    # [5][nz][ny][nx] float64
    t0: float = 0.0
    cfl: float | None = None     # dt = cfl*dx/max_signal_speed, re-evaluated every step
    dt: float | None = None      # fixed dt (config 2)
    nsteps: int = 0
    options: dict = dataclasses.field(default_factory=dict)
    eos_table: tuple | None = None   # (p values on a uniform e grid, e_min, e_max): tabulated closure p(e), eos kind 2


def prim_to_cons(e, n, vx, vy, vz):
    """Definition of the conserved variables (not a hot-path step)."""
    e = np.asarray(e, dtype=np.float64)
    v2 = vx * vx + vy * vy + vz * vz
    g2 = 1.0 / (1.0 - v2)
    p = e / 3.0
    w = (e + p) * g2
    out = np.empty((5,) + e.shape, dtype=np.float64)
    out[0] = w - p
    out[1] = w * vx
    out[2] = w * vy
    out[3] = w * vz
    out[4] = n * np.sqrt(g2)
    return out


def prim_to_cons_p0(e, n, vx, vy, vz, p0):
    """The same definition with the constant-pressure closure p = p0."""
    e = np.asarray(e, dtype=np.float64)
    v2 = vx * vx + vy * vy + vz * vz
    g2 = 1.0 / (1.0 - v2)
    w = (e + p0) * g2
    out = np.empty((5,) + e.shape, dtype=np.float64)
    out[0] = w - p0
    out[1] = w * vx
    out[2] = w * vy
    out[3] = w * vz
    out[4] = n * np.sqrt(g2)
    return out


def crossover_eos_table(n=4096, e_max=64.0, a=0.18, e_c=1.0):
    """A smooth 'crossover' equation of state as a table (input data for the tabulated closure):
    c_s^2(e) = 1/3 - a/(1 + (e/e_c)^2) rises from 1/3 - a at low energy density to 1/3 (the p = e/3 gas) at high,
    p(e) = e/3 - a e_c atan(e/e_c).  Returns (p values at n uniform points of [0, e_max], 0.0, e_max)."""
    e = np.linspace(0.0, e_max, n)
    return e / 3.0 - a * e_c * np.arctan(e / e_c), 0.0, float(e_max)


def cell_centres(n, dx, origin):
    return origin + (np.arange(n, dtype=np.float64) + 0.5) * dx


# ---------------------------------------------------------------- config 1
def sod(nx=400, scheme=WENO5, nsteps=300, cfl=0.25):
    """1+1D relativistic Sod tube (BASELINE.json configs[0]).

    400 cells on [-1,1]; the diaphragm is the face between cells nx/2-1 and nx/2.
    """
    dx = 2.0 / nx
    x = cell_centres(nx, dx, -1.0)
    left = x < 0.0
    e = np.where(left, 10.0, 1.0)
    n = np.where(left, 1.0, 0.1)
    z = np.zeros(nx)
    cons = prim_to_cons(e, n, z, z, z).reshape(5, 1, 1, nx)
    return Workload("sod", (nx, 1, 1), dx, (-1.0, 0.0, 0.0), scheme,
                    (BC_OUTFLOW, BC_OUTFLOW, BC_OUTFLOW), cons, 0.0, cfl=cfl, nsteps=nsteps)


# ---------------------------------------------------------------- configs 2, 3
def hubble_fields(x, y, z, t, t0, e0, n0, axes=(True, True, True), b=(0.0, 0.0, 0.0)):
    """Closed-form d-dimensional Hubble flow for p=e/3.

    v_i = x_i/t on the flagged axes, tau^2 = t^2 - sum x_i^2 over those axes, d = their number,
    e = e0 (t0/tau)^(4d/3), n = n0 (t0/tau)^d exp(-s/2), s = sum (x_i/t)^2/b_i^2 over axes with b_i>0.
    x, y, z broadcastable coordinate arrays.  Returns e, n, vx, vy, vz.
    """
    coords = (x, y, z)
    d = sum(1 for a in axes if a)
    r2 = 0.0
    s = 0.0
    v = []
    for c, a, bi in zip(coords, axes, b):
        if a:
            r2 = r2 + c * c
            v.append(c / t + 0.0 * (x + y + z))
            if bi > 0.0:
                s = s + (c / t) ** 2 / (bi * bi)
        else:
            v.append(0.0 * (x + y + z))
    tau = np.sqrt(t * t - r2) + 0.0 * (x + y + z)
    e = e0 * (t0 / tau) ** (4.0 * d / 3.0)
    n = n0 * (t0 / tau) ** d * np.exp(-0.5 * s)
    return e, n, v[0], v[1], v[2]


def hubble(n=128, half_width=4.0, t0=8.0, scheme=WENO5, nsteps=100, dt_over_dx=0.1):
    """Config 2 with SURVEY reading Q13 (t0 = 8 so the box is inside the light cone)."""
    dx = 2.0 * half_width / n
    c = cell_centres(n, dx, -half_width)
    X, Y, Z = c[None, None, :], c[None, :, None], c[:, None, None]
    e, nn, vx, vy, vz = hubble_fields(X, Y, Z, t0, t0, 1.0, 1.0)
    cons = prim_to_cons(e, nn, vx, vy, vz)
    opts = {"hubble_t0": t0, "hubble_e0": 1.0, "hubble_n0": 1.0}
    return Workload("hubble", (n, n, n), dx, (-half_width,) * 3, scheme,
                    (BC_HUBBLE,) * 3, cons, t0, dt=dt_over_dx * dx, nsteps=nsteps, options=opts)


ELLIPSOID_B = (0.25 * 1.0, 0.25 * 1.3, 0.25 * 1.7)


def ellipsoidal(n=256, half_width=6.0, t0=12.0, scheme=WENO7, nsteps=100, cfl=0.2,
                bc=BC_OUTFLOW):
    """Config 3 with SURVEY reading Q14 (Hubble velocity field, ellipsoidal charge profile)."""
    dx = 2.0 * half_width / n
    c = cell_centres(n, dx, -half_width)
    X, Y, Z = c[None, None, :], c[None, :, None], c[:, None, None]
    e, nn, vx, vy, vz = hubble_fields(X, Y, Z, t0, t0, 1.0, 1.0, b=ELLIPSOID_B)
    cons = prim_to_cons(e, nn, vx, vy, vz)
    opts = {"hubble_t0": t0, "hubble_e0": 1.0, "hubble_n0": 1.0,
            "hubble_bx": ELLIPSOID_B[0], "hubble_by": ELLIPSOID_B[1], "hubble_bz": ELLIPSOID_B[2]}
    return Workload("ellipsoidal", (n, n, n), dx, (-half_width,) * 3, scheme,
                    (bc,) * 3, cons, t0, cfl=cfl, nsteps=nsteps, options=opts)


# ---------------------------------------------------------------- p = const: anisotropic free streaming (ref. [8])
FREE_T = (2.0, 2.6, 3.4)


def free_streaming_cons(x, y, z, t, p0=1.0, Q0=6.0, R0=1.0, T=FREE_T, axes=(True, True, True)):
    """Exact solution for the closure p = p0 (the anisotropic flow of the paper's ref. [8],
    v_i = x_i / (t + T_i), is exact for constant pressure).  Every fluid element moves with constant velocity
    xi_i = x_i / (t + T_i), so Q = E + p0 = (e + p0) gamma^2 and R = n gamma obey the continuity equation, whose
    solution along those straight lines is  Q = G(xi) / J(t),  R = H(xi) / J(t),  J = prod_i (t + T_i) / T_i  over
    the flagged axes; G = Q0 exp(-|xi|^2 / 2), H = R0 exp(-|xi|^2).  Returns the conserved variables
    E = Q - p0, M_i = Q xi_i, R (broadcast arrays)."""
    coords = (x, y, z)
    zero = 0.0 * (x + y + z)
    xi, J, xi2 = [], 1.0, zero
    for c, Ti, a in zip(coords, T, axes):
        if a:
            xi.append(c / (t + Ti) + zero)
            J = J * (t + Ti) / Ti
            xi2 = xi2 + (c / (t + Ti)) ** 2
        else:
            xi.append(zero)
    Q = Q0 * np.exp(-0.5 * xi2) / J
    R = R0 * np.exp(-xi2) / J
    out = np.empty((5,) + np.shape(zero), dtype=np.float64)
    out[0] = Q - p0
    out[1], out[2], out[3] = Q * xi[0], Q * xi[1], Q * xi[2]
    out[4] = R
    return out


def free_streaming(n=48, half_width=1.0, scheme=WENO5, nsteps=40, cfl=0.2, p0=1.0):
    """3-D free-streaming workload for the p = p0 closure on [-L, L]^3 from t = 0, zero-gradient outflow (every
    characteristic speed is v_d, pointing outward at all six faces)."""
    dx = 2.0 * half_width / n
    c = cell_centres(n, dx, -half_width)
    cons = free_streaming_cons(c[None, None, :], c[None, :, None], c[:, None, None], 0.0, p0=p0)
    return Workload("free_streaming", (n, n, n), dx, (-half_width,) * 3, scheme, (BC_OUTFLOW,) * 3, cons, 0.0,
                    cfl=cfl, nsteps=nsteps, options={"eos": 1, "eos_p0": p0})


# ---------------------------------------------------------------- configs 4, 5
def _hotspot_profiles(n, box, centres, sigma):
    """Per-axis Gaussian factors with the minimum-image distance: [3][K][n]."""
    dx = box / n
    c = cell_centres(n, dx, 0.0)
    out = []
    for ax in range(3):
        d = c[None, :] - centres[:, ax][:, None]
        d = d - box * np.round(d / box)
        out.append(np.exp(-0.5 * (d / sigma[:, None]) ** 2))
    return out


def _sum_separable(w, gx, gy, gz):
    """sum_k w_k gz_k[z] gy_k[y] gx_k[x] as one matrix product (the Gaussians are separable)."""
    nz, ny, nx = gz.shape[1], gy.shape[1], gx.shape[1]
    zy = (gz[:, :, None] * gy[:, None, :]).reshape(gz.shape[0], nz * ny)   # [K][nz*ny]
    return (zy.T @ (w[:, None] * gx)).reshape(nz, ny, nx)


def lumpy(n=256, hotspots=40, with_velocity=False, scheme=MUSTA_FORCE, nsteps=50, cfl=0.2,
          box=16.0, seed=SEED, sigma_unit=None, crop=None):
    """Configs 4 (40 hotspots, v=0) and 5 (200 hotspots, per-hotspot velocities, Q15).

    Draw order: all centres, all widths, all amplitudes, then (config 5) speeds and
    directions from normalised Gaussians.  e = 0.1 + sum_k A_k g_k, n = 0.2 e^(3/4),
    v = sum_k A_k g_k v_k / (0.1 + sum_k A_k g_k).  Small parity cases pass a smaller ``box`` and a
    ``sigma_unit`` so that the hotspots span a similar number of cells as at full size.
    ``crop`` = m evaluates only the corner block of the first m cells per axis of the n^3 state (same draws, same
    formulas: the corner crop of the full state up to the summation order of the matrix product), for the CPU
    baseline's bounded sample; the result is a Workload on an m^3 grid.
    """
    rng = np.random.default_rng(seed)
    centres = rng.uniform(0.0, box, size=(hotspots, 3))
    sigma = rng.uniform(0.3, 0.8, size=hotspots) * (box / 16.0 if sigma_unit is None else sigma_unit)
    amp = np.exp(0.5 * rng.standard_normal(hotspots))
    gx, gy, gz = _hotspot_profiles(n, box, centres, sigma)
    if crop is not None:
        gx, gy, gz = gx[:, :crop], gy[:, :crop], gz[:, :crop]
    bump = _sum_separable(amp, gx, gy, gz)
    e = 0.1 + bump
    nn = 0.2 * e ** 0.75
    if with_velocity:
        speed = rng.uniform(0.0, 0.5, size=hotspots)
        dirs = rng.standard_normal((hotspots, 3))
        dirs /= np.linalg.norm(dirs, axis=1)[:, None]
        vk = speed[:, None] * dirs
        v = [_sum_separable(amp * vk[:, a], gx, gy, gz) / e for a in range(3)]
    else:
        v = [np.zeros_like(e)] * 3
    cons = prim_to_cons(e, nn, v[0], v[1], v[2])
    dx = box / n
    name = "lumpy_v" if with_velocity else "lumpy"
    if crop is not None:
        return Workload("%s_crop%d" % (name, crop), (crop, crop, crop), dx, (0.0, 0.0, 0.0), scheme,
                        (BC_PERIODIC,) * 3, cons, 0.0, cfl=cfl, nsteps=nsteps)
    return Workload(name, (n, n, n), dx, (0.0, 0.0, 0.0), scheme, (BC_PERIODIC,) * 3, cons, 0.0,
                    cfl=cfl, nsteps=nsteps)


def production(n=512, scheme=WENO5, nsteps=20):
    """Config 5: the headline case (512^3, 200 hotspots, blended hotspot velocities)."""
    return lumpy(n=n, hotspots=200, with_velocity=True, scheme=scheme, nsteps=nsteps, cfl=0.2)


def random_state(shape, seed, vmax=0.6):
    """Seeded generic admissible state (for unit parity of the kernels): e in [0.5,2], |v|<=vmax."""
    rng = np.random.default_rng(seed)
    e = rng.uniform(0.5, 2.0, size=shape)
    nn = rng.uniform(0.1, 1.0, size=shape)
    sp = rng.uniform(0.0, vmax, size=shape)
    d = rng.standard_normal((3,) + tuple(shape))
    d /= np.sqrt((d * d).sum(axis=0))
    return prim_to_cons(e, nn, sp * d[0], sp * d[1], sp * d[2])
