"""Pins of the oracle's constant-pressure closure p = p0 (the paper's ref. [8] test,
PAPER.md:50).  CPU only; expected values are definitions, numerical eigenvalues and a closed-form solution."""
import math

import numpy as np
import pytest

from paper_1604_03360_b200 import workloads as W

P0 = 0.7


def test_con2prim_round_trip(oracle):
    rng = np.random.default_rng(8)
    for _ in range(200):
        e, n = rng.uniform(0.1, 5.0), rng.uniform(0.1, 2.0)
        sp = rng.uniform(0.0, 0.95)
        d = rng.normal(size=3)
        v = sp * d / np.linalg.norm(d)
        u = W.prim_to_cons_p0(np.array(e), np.array(n), np.array(v[0]), np.array(v[1]), np.array(v[2]), P0)
        got, flag = oracle.con2prim_eos(u, 1, P0)
        assert flag == 0
        g2 = 1.0 / (1.0 - sp * sp)
        assert abs(got[0] - e) <= 1e-13 * (e + P0) * g2 and got[1] == P0
        assert abs(got[2] - n) <= 1e-13 * n * g2 and np.max(np.abs(got[3:] - v)) <= 1e-14
    # the default closure is untouched
    u = W.prim_to_cons(np.array(1.3), np.array(0.4), np.array(0.2), np.array(-0.1), np.array(0.3))
    assert np.array_equal(oracle.con2prim_eos(u, 0, 0.0)[0], oracle.con2prim(u)[0])


def _flux(u, d, p0):
    H = u[0] + p0
    v = u[1:4] / H
    F = np.empty(5)
    F[0] = u[1 + d]
    F[1:4] = u[1:4] * v[d]
    F[1 + d] += p0
    F[4] = u[4] * v[d]
    return F


def test_wave_speed_is_the_flux_jacobian_spectral_radius(oracle):
    """All eigenvalues of dF_d/dU for p = p0 equal v_d (c_s = 0); the Jacobian is formed by central differences of
    the flux written from its definition."""
    rng = np.random.default_rng(9)
    for _ in range(20):
        sp = rng.uniform(0.05, 0.8)
        dvec = rng.normal(size=3)
        v = sp * dvec / np.linalg.norm(dvec)
        u = W.prim_to_cons_p0(np.array(2.0), np.array(0.5), np.array(v[0]), np.array(v[1]), np.array(v[2]), P0)
        for d in range(3):
            J = np.empty((5, 5))
            for k in range(5):
                h = 1e-6 * max(1.0, abs(u[k]))
                up, um = u.copy(), u.copy()
                up[k] += h
                um[k] -= h
                J[:, k] = (_flux(up, d, P0) - _flux(um, d, P0)) / (2 * h)
            lam = np.linalg.eigvals(J)
            assert np.max(np.abs(lam - v[d])) < 1e-3            # a defective eigenvalue: sqrt-of-noise accuracy
            assert abs(oracle.signal_speed(v, d, 1, P0) - abs(v[d])) == 0.0


def _run_free_streaming_1d(oracle, n, scheme, axis=0, T_end=0.5):
    L = 1.0
    dx = 2 * L / n
    c = W.cell_centres(n, dx, -L)
    axes = tuple(a == axis for a in range(3))
    z = np.zeros(1)
    coords = [z[None, None, :], z[None, :, None], z[:, None, None]]
    shape = [1, 1, 1]
    shape[2 - axis] = n
    coords[axis] = c.reshape(shape)
    cons = W.free_streaming_cons(coords[0], coords[1], coords[2], 0.0, p0=1.0, axes=axes)
    nn = [1, 1, 1]
    nn[axis] = n
    o = oracle.Oracle(nn[0], nn[1], nn[2], dx, scheme, eos=1, eos_p0=1.0)
    o.set_state(cons)
    steps = int(round(T_end / (0.2 * dx)))
    o.step(T_end / steps, steps)
    exact = W.free_streaming_cons(coords[0], coords[1], coords[2], T_end, p0=1.0, axes=axes)
    u = o.get_state()
    inner = np.abs(c) <= 0.6
    err = np.abs(u - exact).reshape(5, n)[:, inner]
    return np.max(err[0]) / np.max(np.abs(exact[0])), np.max(err[4]) / np.max(exact[4])


@pytest.mark.parametrize("scheme", [W.WENO5, W.WENO7, W.MUSTA_FORCE])
def test_free_streaming_closed_form_converges(oracle, scheme):
    """Max-norm error on |x| <= 0.6 against the closed form at t = 0.5.  (Measured: WENO5 2.3e-5 -> 7.5e-9,
    WENO7 1.1e-4 -> 6.0e-7, MUSTA-FORCE/minmod 4.5e-5 -> 1.7e-5 from 80 to 160 cells; on coarser grids the
    zero-gradient boundary dominates.)"""
    e1, r1 = _run_free_streaming_1d(oracle, 80, scheme)
    e2, r2 = _run_free_streaming_1d(oracle, 160, scheme)
    assert e2 < e1 and r2 < r1
    assert e2 < {W.WENO5: 5e-8, W.WENO7: 3e-6, W.MUSTA_FORCE: 5e-5}[scheme], (e1, e2)
    order = math.log2(e1 / e2)
    assert order > (1.2 if scheme == W.MUSTA_FORCE else 4.0), (e1, e2, order)


def test_free_streaming_along_each_axis(oracle):
    """The same 1-D solution run along x, y and z (with that axis' T_i) isolates each sweep direction."""
    for axis in range(3):
        e, r = _run_free_streaming_1d(oracle, 80, W.WENO5, axis=axis)
        assert e < 5e-5 and r < 5e-5, (axis, e, r)


def test_uniform_state_and_conservation(oracle):
    u0 = W.prim_to_cons_p0(np.array(1.7), np.array(0.3), np.array(0.31), np.array(-0.22), np.array(0.13), 1.0)
    n = (8, 7, 9)
    u = np.broadcast_to(u0.reshape(5, 1, 1, 1), (5, n[2], n[1], n[0])).copy()
    for scheme in (W.WENO5, W.MUSTA_FORCE):
        o = oracle.Oracle(n[0], n[1], n[2], 0.1, scheme, eos=1, eos_p0=1.0, bc_x=1, bc_y=1, bc_z=1)
        assert np.all(o.eval_L(u) == 0.0)
    w = W.free_streaming(n=12, nsteps=5)
    w.bc = (W.BC_PERIODIC,) * 3
    o = oracle.from_workload(w)
    tot0 = [math.fsum(w.cons[c].ravel()) for c in range(5)]
    oracle.run(o, w)
    tot1 = [math.fsum(o.get_state()[c].ravel()) for c in range(5)]
    for a, b in zip(tot0, tot1):
        assert abs(a - b) <= 1e-13 * tot0[0]
