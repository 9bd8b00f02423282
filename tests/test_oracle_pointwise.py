"""Pins for the oracle's pointwise pieces.  CPU only.

Every expected value here comes from the definitions (T^{mu nu} of an ideal fluid, eigenvalues of
the flux Jacobian built from those definitions), never from the oracle or the CUDA path.
"""
import numpy as np
import pytest

CS2 = 1.0 / 3.0


def prim_to_cons(e, n, v):
    """Definition: E = (e+p)g^2 - p, M = (e+p)g^2 v, R = n g, p = e/3 (SURVEY section 8 notation)."""
    v = np.asarray(v, float)
    g2 = 1.0 / (1.0 - v @ v)
    p = e / 3.0
    w = (e + p) * g2
    return np.array([w - p, w * v[0], w * v[1], w * v[2], n * np.sqrt(g2)])


def flux_from_prim(e, n, v, d):
    """Definition: T^{d0} = M_d, T^{dj} = (e+p)g^2 v_j v_d + p delta_jd, N^d = n g v_d."""
    v = np.asarray(v, float)
    g2 = 1.0 / (1.0 - v @ v)
    p = e / 3.0
    w = (e + p) * g2
    F = np.array([w * v[d], w * v[0] * v[d], w * v[1] * v[d], w * v[2] * v[d], n * np.sqrt(g2) * v[d]])
    F[1 + d] += p
    return F


def random_prims(rng, vmax, count):
    for _ in range(count):
        e = rng.uniform(0.05, 20.0)
        n = rng.uniform(0.01, 5.0)
        d = rng.standard_normal(3)
        v = rng.uniform(0.0, vmax) * d / np.linalg.norm(d)
        yield e, n, v


# ------------------------------------------------------------------ O1 con2prim
@pytest.mark.parametrize("vmax,tol", [(0.9, 2e-14), (0.995, 5e-13)])
def test_con2prim_round_trip(oracle, vmax, tol):
    rng = np.random.default_rng(11)
    worst = 0.0
    for e, n, v in random_prims(rng, vmax, 2000):
        out, flag = oracle.con2prim(prim_to_cons(e, n, v))
        assert flag == 0
        ref = np.array([e, e / 3.0, n, *v])
        scale = np.array([e, e, n, 1.0, 1.0, 1.0])
        worst = max(worst, np.max(np.abs(out - ref) / scale))
    assert worst < tol, worst


def test_con2prim_at_rest_is_exact(oracle):
    out, flag = oracle.con2prim([3.0, 0.0, 0.0, 0.0, 0.7])
    assert flag == 0
    assert np.allclose(out, [3.0, 1.0, 0.7, 0, 0, 0], rtol=0, atol=1e-15)


def test_con2prim_single_axis_matches_quadratic(oracle):
    # 1D: |M| v^2 - 4 E v + 3|M| = 0 -> v = (2E - sqrt(4E^2-3M^2))/M on each axis alone
    for ax in range(3):
        u = np.zeros(5)
        u[0], u[1 + ax], u[4] = 2.0, -1.3, 0.4
        out, _ = oracle.con2prim(u)
        v = (2 * 2.0 - np.sqrt(4 * 4.0 - 3 * 1.69)) / (-1.3)
        assert abs(out[3 + ax] - v) < 1e-15
        assert abs(out[0] - (2.0 - (-1.3) * v)) < 1e-14          # e = E - M.v
        others = [3 + a for a in range(3) if a != ax]
        assert np.all(out[others] == 0.0)


def test_con2prim_unphysical_flag(oracle):
    # Q16: |M| > E is clamped and flagged; E <= 0 is flagged
    _, flag = oracle.con2prim([1.0, 2.0, 0.0, 0.0, 0.1])
    assert flag == 1
    out, flag = oracle.con2prim([-1.0, 0.0, 0.0, 0.0, 0.1])
    assert flag == 1 and np.all(np.isfinite(out))


# ------------------------------------------------------------------ a5 physical flux
def test_phys_flux_matches_energy_momentum_tensor(oracle):
    rng = np.random.default_rng(12)
    for e, n, v in random_prims(rng, 0.95, 300):
        u = prim_to_cons(e, n, v)
        for d in range(3):
            F = oracle.phys_flux(u, d)
            ref = flux_from_prim(e, n, v, d)
            assert np.max(np.abs(F - ref)) < 2e-13 * np.max(np.abs(u)), (F, ref)


# ------------------------------------------------------------------ O2 wave speeds
def _jacobian_eigs(e, n, v, d):
    """Eigenvalues of dF_d/dU = (dF/dW)(dU/dW)^-1, W = (e, n, v) by central differences of the
    *definitions* above."""
    W0 = np.array([e, n, *v])
    A = np.empty((5, 5))
    B = np.empty((5, 5))
    for k in range(5):
        h = 1e-6 * max(1.0, abs(W0[k]))
        Wp, Wm = W0.copy(), W0.copy()
        Wp[k] += h
        Wm[k] -= h
        A[:, k] = (flux_from_prim(Wp[0], Wp[1], Wp[2:], d) - flux_from_prim(Wm[0], Wm[1], Wm[2:], d)) / (2 * h)
        B[:, k] = (prim_to_cons(Wp[0], Wp[1], Wp[2:]) - prim_to_cons(Wm[0], Wm[1], Wm[2:])) / (2 * h)
    lam = np.linalg.eigvals(A @ np.linalg.inv(B))
    assert np.max(np.abs(lam.imag)) < 1e-5
    return np.sort(lam.real)


def test_signal_speed_is_spectral_radius_of_flux_jacobian(oracle):
    rng = np.random.default_rng(13)
    for e, n, v in random_prims(rng, 0.9, 200):
        for d in range(3):
            lam = _jacobian_eigs(e, n, v, d)
            a = oracle.signal_speed(v, d)
            assert abs(a - max(abs(lam[0]), abs(lam[-1]))) < 2e-7, (a, lam)
            assert np.allclose(lam[1:4], v[d], atol=2e-6)          # triple eigenvalue v_d
            assert 0.0 < a < 1.0


def test_signal_speed_special_cases(oracle):
    cs = np.sqrt(CS2)
    for d in range(3):
        assert abs(oracle.signal_speed([0, 0, 0], d) - cs) < 1e-16
    # 1D relativistic velocity addition (|v_d| + c_s)/(1 + |v_d| c_s)
    for vd in (-0.8, -0.2, 0.3, 0.95):
        for d in range(3):
            v = [0.0, 0.0, 0.0]
            v[d] = vd
            assert abs(oracle.signal_speed(v, d) - (abs(vd) + cs) / (1 + abs(vd) * cs)) < 2e-15
    # purely transverse motion: lambda = +- c_s sqrt(1-v^2) / sqrt(1 - v^2 c_s^2) ... from the O2 formula
    vt = 0.6
    expect = cs * np.sqrt((1 - vt * vt) * (1 - vt * vt * CS2)) / (1 - vt * vt * CS2)
    assert abs(oracle.signal_speed([0.0, vt, 0.0], 0) - expect) < 1e-15


# ------------------------------------------------------------------ O6 minmod
def test_minmod_truth_table(oracle):
    assert oracle.minmod(1.0, 2.0) == 1.0
    assert oracle.minmod(3.0, 2.0) == 2.0
    assert oracle.minmod(-1.0, -2.0) == -1.0
    assert oracle.minmod(-3.0, -2.0) == -2.0
    assert oracle.minmod(1.0, -2.0) == 0.0
    assert oracle.minmod(-1.0, 2.0) == 0.0
    assert oracle.minmod(0.0, 2.0) == 0.0
    assert oracle.minmod(2.0, 0.0) == 0.0
