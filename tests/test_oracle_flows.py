"""Whole-solver pins of the oracle against the mathematics, part 2: the paper's two 3+1D
validation flows ("ellipsoidal flow solution [8] and Hubble-like solution were done in full 3+1D") with
the analytic ghost fill and its stage times, the zero-gradient outflow rule, MUSTA-FORCE's wave-speed choice,
measured orders of accuracy ("second (MUSTA-FORCE), fifth and seventh (WENO) order"), symmetries, and an
isentropic simple wave.  CPU only; nothing here is compared with the CUDA path.

The closed forms used as expected values (workloads.hubble_fields, workloads.free_streaming_cons) are themselves
pinned to Eq. (1) first, by a finite-difference residual of the conservation laws."""
import math

import numpy as np
import pytest

from paper_1604_03360_b200 import workloads as W

CS = 1.0 / math.sqrt(3.0)


def d4(f, h):
    """4th-order central difference of f at 0."""
    return (-f(2 * h) + 8 * f(h) - 8 * f(-h) + f(-2 * h)) / (12 * h)


# ------------------------------------------------------------------ (d) the closed forms solve Eq. (1)
def _hubble_cons_and_fluxes(t, x, y, z, axes, b):
    e, n, vx, vy, vz = W.hubble_fields(np.float64(x), np.float64(y), np.float64(z), t, 8.0, 1.3, 0.7, axes=axes, b=b)
    v = np.array([vx, vy, vz], dtype=float)
    p = e / 3.0
    g2 = 1.0 / (1.0 - v @ v)
    w = (e + p) * g2
    U = np.array([w - p, w * v[0], w * v[1], w * v[2], n * math.sqrt(g2)])
    # T^{i nu}, N^i (SURVEY section 8 notation): F^i_E = M_i, F^i_{M_j} = M_j v_i + p delta_ij, F^i_R = R v_i
    F = [np.array([U[1 + i], U[1] * v[i] + (p if i == 0 else 0), U[2] * v[i] + (p if i == 1 else 0),
                   U[3] * v[i] + (p if i == 2 else 0), U[4] * v[i]]) for i in range(3)]
    return U, F


@pytest.mark.parametrize("axes,b", [((True, False, False), (0, 0, 0)), ((False, True, True), (0, 0, 0)),
                                    ((True, True, True), (0, 0, 0)), ((True, True, True), W.ELLIPSOID_B),
                                    ((True, False, True), (0.3, 0, 0.5))])
def test_hubble_closed_form_satisfies_the_conservation_laws(axes, b):
    """dU/dt + sum_i dF_i/dx_i = 0 (Eq. 1) at scattered points, derivatives by central differences."""
    rng = np.random.default_rng(5)
    h = 2e-3
    for _ in range(6):
        t = rng.uniform(8.0, 9.0)
        pt = rng.uniform(-3.0, 3.0, size=3) * np.array(axes, dtype=float)
        res = d4(lambda s: _hubble_cons_and_fluxes(t + s, pt[0], pt[1], pt[2], axes, b)[0], h)
        scale = np.abs(res).copy()
        for i in range(3):
            def Fi(s, i=i):
                q = pt.copy()
                q[i] += s
                return _hubble_cons_and_fluxes(t, q[0], q[1], q[2], axes, b)[1][i]
            term = d4(Fi, h)
            res = res + term
            scale = np.maximum(scale, np.abs(term))
        assert np.all(np.abs(res) <= 1e-9 * np.maximum(scale, 1e-3)), (axes, b, res, scale)


def test_free_streaming_closed_form_satisfies_the_conservation_laws():
    """The p = p0 solution of ref. [8]: same residual test with the constant-pressure flux."""
    rng = np.random.default_rng(6)
    h, p0 = 2e-3, 1.0

    def UF(t, q):
        U = W.free_streaming_cons(np.float64(q[0]), np.float64(q[1]), np.float64(q[2]), t, p0=p0)
        v = U[1:4] / (U[0] + p0)
        F = [np.array([U[1 + i], U[1] * v[i] + (p0 if i == 0 else 0), U[2] * v[i] + (p0 if i == 1 else 0),
                       U[3] * v[i] + (p0 if i == 2 else 0), U[4] * v[i]]) for i in range(3)]
        return U, F
    for _ in range(6):
        t = rng.uniform(0.0, 1.0)
        pt = rng.uniform(-1.0, 1.0, size=3)
        res = d4(lambda s: UF(t + s, pt)[0], h)
        scale = np.abs(res).copy()
        for i in range(3):
            def Fi(s, i=i):
                q = pt.copy()
                q[i] += s
                return UF(t, q)[1][i]
            term = d4(Fi, h)
            res, scale = res + term, np.maximum(scale, np.abs(term))
        assert np.all(np.abs(res) <= 1e-9 * np.maximum(scale, 1e-3)), (res, scale)


# ------------------------------------------------------------------ (a) Hubble flows with analytic ghosts
def hubble_workload(n, axes, scheme, nsteps, half=4.0, t0=8.0, b=(0.0, 0.0, 0.0), dt_over_dx=0.1, bc=W.BC_HUBBLE):
    """d-dimensional Hubble flow on the flagged axes (n cells each, the others inactive), SURVEY O9 / Q13 / Q14."""
    dx = 2.0 * half / n
    c = W.cell_centres(n, dx, -half)
    one = np.zeros(1)
    X = (c if axes[0] else one)[None, None, :]
    Y = (c if axes[1] else one)[None, :, None]
    Z = (c if axes[2] else one)[:, None, None]
    e, nn, vx, vy, vz = W.hubble_fields(X, Y, Z, t0, t0, 1.0, 1.0, axes=axes, b=b)
    cons = W.prim_to_cons(e, nn, vx, vy, vz)
    shape = tuple(n if a else 1 for a in axes)
    opts = {"hubble_t0": t0, "hubble_e0": 1.0, "hubble_n0": 1.0, "hubble_bx": b[0], "hubble_by": b[1], "hubble_bz": b[2]}
    w = W.Workload("hubble_d", shape, dx, tuple(-half if a else 0.0 for a in axes), scheme,
                   tuple(bc if a else W.BC_OUTFLOW for a in axes), cons, t0, dt=dt_over_dx * dx, nsteps=nsteps,
                   options=opts)
    return w, (X, Y, Z)


def run_against_closed_form(oracle, w, coords, axes, b=(0.0, 0.0, 0.0), t0=8.0):
    o = oracle.from_workload(w)
    oracle.run(o, w)
    t = o.time
    e, nn, vx, vy, vz = W.hubble_fields(coords[0], coords[1], coords[2], t, t0, 1.0, 1.0, axes=axes, b=b)
    exact = W.prim_to_cons(e, nn, vx, vy, vz)
    u = o.get_state()
    assert abs(t - (t0 + w.nsteps * w.dt)) < 1e-12
    return u, exact


# measured with the oracle as committed (max abs error after 20 steps at n = 32); thresholds are 1.5x these.  A ghost
# fill at the wrong stage time (t + dt instead of t + dt/2 in stage 3) gives 3e-4, a wrong exponent 1e-2.
BJORKEN_ERR = {W.WENO5: 1.05e-5, W.WENO7: 6.4e-7, W.MUSTA_FORCE: 1.53e-3}


@pytest.mark.parametrize("scheme", [W.WENO5, W.WENO7, W.MUSTA_FORCE])
def test_bjorken_flow_along_each_axis_matches_the_closed_form_and_permutes(oracle, scheme):
    """d = 1 Hubble ("Bjorken") flow along x, y and z in turn with analytic ghosts (BC_HUBBLE): e ~ tau^(-4/3),
    n ~ 1/tau.  Pins hubble_cons for d = 1, the analytic fill, the stage times t, t+dt, t+dt/2 (O8), and isolates
    each sweep direction: the three runs must be axis permutations of each other."""
    outs = []
    for axis in range(3):
        axes = tuple(a == axis for a in range(3))
        w, coords = hubble_workload(32, axes, scheme, 20)
        u, exact = run_against_closed_form(oracle, w, coords, axes)
        err = np.max(np.abs(u - exact))
        assert err <= 1.5 * BJORKEN_ERR[scheme], (axis, err)
        assert err >= 0.2 * BJORKEN_ERR[scheme]          # the flow really evolved and the number is not stale
        for other in range(3):
            if other != axis:
                assert np.all(u[1 + other] == 0.0)
        outs.append(np.stack([u[0].ravel(), u[1 + axis].ravel(), u[4].ravel()]))
    assert np.max(np.abs(outs[0] - outs[1])) <= 1e-14 and np.max(np.abs(outs[0] - outs[2])) <= 1e-14


def test_two_dimensional_hubble_flow(oracle):
    """d = 2: e ~ tau^(-8/3), n ~ tau^(-2) (the exponent 4d/3 differs from both d = 1 and d = 3)."""
    errs = {}
    for axes in ((True, True, False), (False, True, True)):
        w, coords = hubble_workload(16, axes, W.WENO5, 10)
        u, exact = run_against_closed_form(oracle, w, coords, axes)
        errs[axes] = np.max(np.abs(u - exact) / np.max(np.abs(exact[0])))
        assert errs[axes] < 1.05e-3, errs        # measured 6.96e-4 (16 cells per axis); threshold 1.5x
    assert abs(errs[(True, True, False)] - errs[(False, True, True)]) < 1e-13


def _hubble3d_errors(oracle, w, t0, b, half, inner_half):
    """(max rel error of E on the whole box, on the inner box, mean rel error of E, max error of R / max R inner)."""
    o = oracle.from_workload(w)
    oracle.run(o, w)
    n = w.n[0]
    c = W.cell_centres(n, w.dx, -half)
    e, nn, vx, vy, vz = W.hubble_fields(c[None, None, :], c[None, :, None], c[:, None, None], o.time, t0, 1.0, 1.0, b=b)
    exact = W.prim_to_cons(e, nn, vx, vy, vz)
    u = o.get_state()
    rel = np.abs(u[0] - exact[0]) / exact[0]
    inner = np.abs(c) <= inner_half
    sel = np.ix_(inner, inner, inner)
    return rel.max(), rel[sel].max(), rel.mean(), np.max(np.abs(u[4] - exact[4])[sel]) / np.max(exact[4]), o.time


def test_config2_reduced_against_the_closed_form(oracle):
    """BASELINE configs[1] at 24^3 (same box, t0 = 8, dt = 0.1 dx, analytic ghosts): d = 3, e ~ tau^-4.  Thresholds
    are 1.5x the oracle's measured errors (E, relative: WENO5 1.36e-3, WENO7 3.85e-3 at the corners, where |v| = 0.87
    and 24 cells per axis do not resolve tau^-4; 2.1e-5 and 3.1e-7 on |x_i| <= 2)."""
    r5 = _hubble3d_errors(oracle, W.hubble(n=24, scheme=W.WENO5, nsteps=12), 8.0, (0, 0, 0), 4.0, 2.0)
    r7 = _hubble3d_errors(oracle, W.hubble(n=24, scheme=W.WENO7, nsteps=12), 8.0, (0, 0, 0), 4.0, 2.0)
    assert abs(r5[4] - (8.0 + 12 * 0.1 * 8.0 / 24)) < 1e-12
    assert 0.3 * 1.36e-3 < r5[0] < 1.5 * 1.36e-3 and r5[1] < 1.5 * 2.13e-5, r5
    assert r7[0] < 1.5 * 3.85e-3 and r7[1] < 1.5 * 3.1e-7, r7
    # PAPER.md:50 "higher order simulations were slightly more accurate": where the flow is resolved, and on average
    assert r7[1] < r5[1] and r7[2] < r5[2]


@pytest.mark.parametrize("bc", [W.BC_HUBBLE, W.BC_OUTFLOW])
def test_config3_reduced_against_the_closed_form(oracle, bc):
    """BASELINE configs[2] at 24^3 (reading Q14: Hubble velocity field with the ellipsoidal charge profile, t0 = 12):
    with the analytic fill everywhere, and with the config's zero-gradient outflow on the part of the box the
    boundary cannot have reached in 6 steps.  Pins the exp(-sigma/2) factor of the charge."""
    res = {}
    for scheme in (W.WENO5, W.WENO7):
        w = W.ellipsoidal(n=24, scheme=scheme, nsteps=6, bc=bc)
        w.cfl, w.dt = None, 0.1 * w.dx
        res[scheme] = _hubble3d_errors(oracle, w, 12.0, W.ELLIPSOID_B, 6.0, 2.0)
    r5, r7 = res[W.WENO5], res[W.WENO7]
    # measured on |x_i| <= 2: E 5.1e-6 (WENO5), 7e-8 (WENO7); R 5.8e-6, 4.9e-7 of max R
    assert r5[1] < 1.5 * 5.1e-6 and r5[3] < 1.5 * 5.8e-6, r5
    assert r7[1] < 1.5 * 7.1e-8 and r7[3] < 1.5 * 4.9e-7, r7
    if bc == W.BC_HUBBLE:   # whole box: 6.2e-4 / 2.2e-3 at the corners
        assert 0.3 * 6.2e-4 < r5[0] < 1.5 * 6.2e-4 and r7[0] < 1.5 * 2.2e-3, (r5, r7)
    else:                   # the zero-gradient boundary is wrong by O(1) for this flow, and must be seen to be
        assert r5[0] > 0.05


# ------------------------------------------------------------------ (b) the zero-gradient outflow rule (Q9)
@pytest.mark.parametrize("scheme,g", [(W.WENO5, 3), (W.WENO7, 4), (W.MUSTA_FORCE, 2)])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_outflow_ghosts_repeat_the_boundary_cell(oracle, scheme, g, axis):
    """L(u) with outflow ghosts must equal, bit for bit, L of the array extended BY HAND with g copies of each
    boundary cell (the definition of zero-gradient ghosts) evaluated where that array's own boundary rule cannot
    matter."""
    n = 12
    shape = [1, 1, 1]
    shape[axis] = n
    u = W.random_state(tuple(reversed(shape)), seed=21, vmax=0.4)          # [5][nz][ny][nx]
    ax = 3 - axis                                                            # array axis of the grid axis
    lo = np.take(u, [0], axis=ax)
    hi = np.take(u, [n - 1], axis=ax)
    ext = np.concatenate([lo] * g + [u] + [hi] * g, axis=ax)
    o = oracle.Oracle(shape[0], shape[1], shape[2], 0.1, scheme)
    L = o.eval_L(u)
    eshape = list(shape)
    eshape[axis] = n + 2 * g
    oe = oracle.Oracle(eshape[0], eshape[1], eshape[2], 0.1, scheme)
    oe.set_option("bc_" + "xyz"[axis], W.BC_PERIODIC)                        # any rule: the middle cannot see it
    Le = np.take(oe.eval_L(ext), range(g, g + n), axis=ax)
    assert np.array_equal(L, Le)
    assert np.max(np.abs(np.take(L, [0, n - 1], axis=ax))) > 0.1             # the boundary cells are not idle


# ------------------------------------------------------------------ (c) MUSTA-FORCE from the FORCE definition (Q7)
def _force_flux(oracle, QL, QR, d, C):
    """FORCE = the mean of the Lax-Friedrichs and the two-step Lax-Wendroff (Richtmyer) fluxes for the local step
    tau = C / max(a_d(QL), a_d(QR)) (reading Q7), from the pinned pointwise pieces."""
    def speed(Q):
        prim, _ = oracle.con2prim(Q)
        return oracle.signal_speed(prim[3:6], d)
    tau = C / max(speed(QL), speed(QR))
    FL, FR = oracle.phys_flux(QL, d), oracle.phys_flux(QR, d)
    lf = 0.5 * (FL + FR) - 0.5 / tau * (QR - QL)
    lw = oracle.phys_flux(0.5 * (QL + QR) - 0.5 * tau * (FR - FL), d)
    return 0.5 * (lf + lw), FL, FR, tau


@pytest.mark.parametrize("d", [0, 1, 2])
def test_musta_force_flux_with_different_velocities_on_the_two_sides(oracle, d):
    """Piecewise-constant data (slopes vanish, Q_L = u_i, Q_R = u_{i+1}) whose two sides move differently, so that
    a_d(Q_L) != a_d(Q_R) and the choice S = max matters.  K = 1 is the FORCE flux; K = 2 applies one corrector
    Q_L <- Q_L - tau (F* - F_L), Q_R <- Q_R - tau (F_R - F*) and evaluates FORCE again (O7)."""
    vl, vr = np.zeros(3), np.zeros(3)
    vl[d], vr[d] = 0.55, -0.15
    vl[(d + 1) % 3], vr[(d + 2) % 3] = 0.2, 0.3
    UL = W.prim_to_cons(np.float64(2.0), np.float64(0.8), *[np.float64(x) for x in vl])
    UR = W.prim_to_cons(np.float64(0.9), np.float64(0.3), *[np.float64(x) for x in vr])
    cells = np.array([UL, UL, UR, UR])
    pl, _ = oracle.con2prim(UL)
    pr, _ = oracle.con2prim(UR)
    aL, aR = oracle.signal_speed(pl[3:6], d), oracle.signal_speed(pr[3:6], d)
    assert abs(aL - aR) > 0.15                                                 # max and min really differ
    f1, FL, FR, tau = _force_flux(oracle, UL, UR, d, 0.9)
    got1 = oracle.musta_force_flux(cells, d, K=1, C=0.9)
    assert np.max(np.abs(got1 - f1)) <= 4e-15 * np.max(np.abs(f1))
    QL2, QR2 = UL - tau * (f1 - FL), UR - tau * (FR - f1)
    f2, *_ = _force_flux(oracle, QL2, QR2, d, 0.9)
    got2 = oracle.musta_force_flux(cells, d, K=2, C=0.9)
    assert np.max(np.abs(got2 - f2)) <= 8e-15 * np.max(np.abs(f2))
    assert np.max(np.abs(f2 - f1)) > 1e-3 * np.max(np.abs(f1))               # the second stage changes the flux


# ------------------------------------------------------------------ (e) measured orders of accuracy
def _advect_error(oracle, scheme, n, axis, t_end, dt):
    """Charge advection: uniform e, v; n(x,0) smooth periodic -> n(x - v t); E, M stay uniform."""
    v = np.zeros(3)
    v[axis] = 0.4
    v[(axis + 1) % 3] = 0.2
    shape = [1, 1, 1]
    shape[axis] = n
    x = W.cell_centres(n, 1.0 / n, 0.0)
    prof = lambda s: 1.0 + 0.3 * np.sin(2 * np.pi * s) + 0.1 * np.cos(4 * np.pi * s)
    ones = np.ones(n)
    u = W.prim_to_cons(1.5 * ones, prof(x), v[0] * ones, v[1] * ones, v[2] * ones)
    o = oracle.Oracle(shape[0], shape[1], shape[2], 1.0 / n, scheme)
    o.set_option("bc_" + "xyz"[axis], W.BC_PERIODIC)
    o.set_state(u.reshape(5, shape[2], shape[1], shape[0]))
    steps = int(round(t_end / dt))
    o.step(t_end / steps, steps)
    out = o.get_state().reshape(5, n)
    gam = 1.0 / math.sqrt(1.0 - v @ v)
    exact = prof(x - v[axis] * t_end) * gam
    assert np.max(np.abs(out[:4] - u[:4])) < 1e-13                            # E and M stay uniform
    return np.sum(np.abs(out[4] - exact)) / n


@pytest.mark.parametrize("scheme,lo,hi,n1,n2", [(W.WENO5, 4.6, 5.5, 32, 64), (W.WENO7, 6.5, 8.3, 32, 48),
                                                 (W.MUSTA_FORCE, 1.6, 2.4, 80, 160)])
def test_charge_advection_has_the_stated_order(oracle, scheme, lo, hi, n1, n2):
    """PAPER.md:7 "second (MUSTA-FORCE), fifth and seventh (WENO) order of accuracy": L1 error of the advected
    charge at two resolutions, with a time step small enough that the RK3 error does not mask the spatial one
    (measured 5.04 / 7.48 / 1.80)."""
    t_end = 0.25
    errs = []
    for n in (n1, n2):
        p = {W.WENO5: 5.0, W.WENO7: 7.0, W.MUSTA_FORCE: 2.0}[scheme]
        dt = 0.3 * (1.0 / n) ** (p / 3.0) / 4.0 if scheme != W.MUSTA_FORCE else 0.2 / n
        errs.append(_advect_error(oracle, scheme, n, 0, t_end, dt))
    order = math.log(errs[0] / errs[1]) / math.log(n2 / n1)
    assert lo < order < hi, (errs, order)


def test_charge_advection_is_the_same_along_every_axis(oracle):
    e = [_advect_error(oracle, W.WENO5, 16, axis, 0.1, 0.004) for axis in range(3)]
    assert abs(e[0] - e[1]) < 1e-15 and abs(e[0] - e[2]) < 1e-15


# ------------------------------------------------------------------ (e) isentropic simple wave
def _simple_wave_exact(x, t, e_of):
    """Right-going simple wave with J_- = artanh v - (sqrt(3)/4) ln e = 0: e, v are constant along
    x = x0 + lambda_+(x0) t, lambda_+ = (v + c_s)/(1 + v c_s); n = e^(3/4) (isentropic).  Periodic in [0, 1)."""
    x0 = x.copy()
    for _ in range(200):
        e0 = e_of(x0)
        v0 = np.tanh(math.sqrt(3.0) / 4.0 * np.log(e0))
        lam = (v0 + CS) / (1.0 + v0 * CS)
        x0 = x - lam * t
    e0 = e_of(x0)
    v0 = np.tanh(math.sqrt(3.0) / 4.0 * np.log(e0))
    assert np.max(np.abs(x0 + (v0 + CS) / (1.0 + v0 * CS) * t - x)) < 1e-14
    return e0, v0, e0 ** 0.75


@pytest.mark.parametrize("scheme,lo", [(W.WENO5, 4.5), (W.WENO7, 6.0)])
def test_isentropic_simple_wave_converges_at_the_design_order(oracle, scheme, lo):
    """Coupled E-M system with a non-trivial pressure: the exact solution follows from the Riemann
    invariant; valid until the characteristics cross (t_b ~ 5 here, the run stops at 0.2)."""
    e_of = lambda s: 1.0 + 0.1 * np.sin(2 * np.pi * s)
    t_end, errs = 0.2, []
    p = 5.0 if scheme == W.WENO5 else 7.0
    for n in (16, 32):
        x = W.cell_centres(n, 1.0 / n, 0.0)
        e0, v0, n0 = _simple_wave_exact(x, 0.0, e_of)
        z = np.zeros(n)
        u = W.prim_to_cons(e0, n0, v0, z, z)
        o = oracle.Oracle(n, 1, 1, 1.0 / n, scheme)
        o.set_option("bc_x", W.BC_PERIODIC)
        o.set_state(u.reshape(5, 1, 1, n))
        steps = int(round(t_end / (0.1 * (1.0 / n) ** (p / 3.0))))
        o.step(t_end / steps, steps)
        ee, ve, ne = _simple_wave_exact(x, t_end, e_of)
        exact = W.prim_to_cons(ee, ne, ve, z, z)
        out = o.get_state().reshape(5, n)
        errs.append(np.sum(np.abs(out - exact)) / n)
    order = math.log2(errs[0] / errs[1])
    assert order > lo, (errs, order)


# ------------------------------------------------------------------ (e) symmetries
@pytest.mark.parametrize("scheme", [W.WENO5, W.WENO7, W.MUSTA_FORCE])
def test_axis_permutation_and_mirror_symmetry(oracle, scheme):
    """Permuting the axes of the data permutes the result; data even in x (M_x odd) stays so.  Not bit-exact: the
    sum over directions is not associative (<= 1e-13)."""
    n = 10
    w = W.lumpy(n=n, hotspots=5, with_velocity=True, scheme=scheme, box=1.5, sigma_unit=0.35, seed=77)
    u = w.cons                                                   # [5][z][y][x]
    dt = 0.1 * w.dx

    def run(state):
        o = oracle.Oracle(n, n, n, w.dx, scheme)
        for ax in "xyz":
            o.set_option("bc_" + ax, W.BC_PERIODIC)
        o.set_state(np.ascontiguousarray(state))
        o.step(dt, 3)
        return o.get_state()
    base = run(u)
    # new x = old y, new y = old z, new z = old x
    perm = np.transpose(u, (0, 1 + 2, 1 + 0, 1 + 1))              # [z'][y'][x'] = [x][z][y]
    perm = perm[[0, 2, 3, 1, 4]]                                  # M_x' = M_y, M_y' = M_z, M_z' = M_x
    got = run(perm)
    back = np.transpose(got[[0, 3, 1, 2, 4]], (0, 2, 3, 1))
    scale = np.max(np.abs(base[0]))
    assert np.max(np.abs(back - base)) <= 1e-13 * scale
    assert np.max(np.abs(base - u)) > 1e-3 * scale
    # mirror in x: x -> -x, M_x -> -M_x
    mir = u[:, :, :, ::-1].copy()
    mir[1] *= -1.0
    gm = run(mir)
    gm = gm[:, :, :, ::-1].copy()
    gm[1] *= -1.0
    assert np.max(np.abs(gm - base)) <= 1e-13 * scale


# ------------------------------------------------------------------ a4 / Q16 details
def test_max_signal_speed_counts_active_axes_only(oracle):
    """A fast flow along y on a grid whose y axis is inactive (ny = 1) must not enter the CFL maximum (a4)."""
    n = 9
    rng = np.random.default_rng(3)
    vx, vz = rng.uniform(-0.2, 0.2, n * n), rng.uniform(-0.2, 0.2, n * n)
    vy = np.full(n * n, 0.9)
    u = W.prim_to_cons(np.full(n * n, 1.0), np.full(n * n, 1.0), vx, vy, vz).reshape(5, n, 1, n)
    o = oracle.Oracle(n, 1, n, 0.1, W.WENO5)
    o.set_state(u)
    expect = 0.0
    for i in range(n * n):
        v = np.array([vx[i], vy[i], vz[i]])
        v2 = v @ v
        for d in (0, 2):
            a = (abs(v[d]) * (2 / 3) + CS * math.sqrt((1 - v2) * (1 - v[d] ** 2 - (v2 - v[d] ** 2) / 3))) / (1 - v2 / 3)
            expect = max(expect, a)
    assert abs(o.max_signal_speed() - expect) < 1e-14
    all_axes = oracle.signal_speed([vx[0], vy[0], vz[0]], 1)
    assert all_axes > expect + 0.1                                # the y speed would have dominated


def test_q16_clamp_values(oracle):
    """Q16: |M| > (1 - 1e-12) E is scaled back to exactly (1 - 1e-12) E along M; E < 1e-300 is raised to 1e-300."""
    E = 2.0
    Mdir = np.array([0.6, -0.64, 0.48])
    Mdir /= np.linalg.norm(Mdir)
    bad, flag = oracle.con2prim(np.array([E, *(1.7 * E * Mdir), 0.3]))
    assert flag == 1
    lim = (1.0 - 1e-12) * E
    ref, flag_ref = oracle.con2prim(np.array([E, *(lim * (1 - 1e-15) * Mdir), 0.3]))   # just inside: not clamped
    assert flag_ref == 0
    assert np.max(np.abs(bad[3:6] - ref[3:6])) < 1e-12 and abs(np.linalg.norm(bad[3:6]) - 1.0) < 1e-11
    assert np.allclose(bad[3:6] / np.linalg.norm(bad[3:6]), Mdir, atol=1e-12)
    assert abs(bad[0] - ref[0]) <= 1e-3 * abs(ref[0]) + 1e-14 and 0 < bad[0] < 1e-10 * E
    low, flag = oracle.con2prim(np.array([0.0, 0.0, 0.0, 0.0, 0.0]))
    assert flag == 1 and 0.0 <= low[0] <= 1e-300 and np.all(low[3:6] == 0.0)       # E raised to the floor, fluid at rest
    neg, flag = oracle.con2prim(np.array([-1.0, 0.1, 0.0, 0.0, 1.0]))
    assert flag == 1                                                               # a negative energy is flagged
