"""Pins for the oracle's interface fluxes: WENO5/7 (O3, O4), LLF split (O5), MUSTA-FORCE (O7).
CPU only.  Expected values: the WENO *definition* evaluated in exact rationals (tests/exact.py),
closed forms for scalar advection, and consistency identities."""
from fractions import Fraction

import numpy as np
import pytest

import exact
from test_oracle_pointwise import prim_to_cons, flux_from_prim


# ------------------------------------------------------------------ O3 / O4 WENO
@pytest.mark.parametrize("r", [3, 4])
def test_weno_matches_definition_in_exact_rationals(oracle, r):
    rng = np.random.default_rng(20 + r)
    fn = oracle.weno5 if r == 3 else oracle.weno7
    for trial in range(12):
        f = [Fraction(int(x), 16) for x in rng.integers(-64, 64, size=2 * r - 1)]
        if trial % 3 == 0:   # a step inside the stencil: strongly nonlinear weights
            f = [Fraction(1)] * r + [Fraction(0)] * (r - 1)
            f[trial % r] += Fraction(trial, 7)
        for eps in (Fraction(1, 10 ** 6), Fraction(1, 100)):
            ref, parts = exact.weno_exact(f, eps)
            got = fn([float(x) for x in f], float(eps))
            assert abs(got - float(ref)) <= 4e-14 * max(1.0, max(abs(float(x)) for x in f)), (f, got, float(ref))


def test_weno_definition_reproduces_the_printed_coefficients():
    """SURVEY O3/O4 coefficient tables equal the definition (guards tests/exact.py itself)."""
    f5 = [Fraction(x) for x in (3, -1, 4, 1, -5)]
    _, p = exact.weno_exact(f5, Fraction(1, 10 ** 6))
    a, b, c, d, e = f5
    assert p["d"] == [Fraction(1, 10), Fraction(6, 10), Fraction(3, 10)]
    assert p["q"] == [(2 * a - 7 * b + 11 * c) / 6, (-b + 5 * c + 2 * d) / 6, (2 * c + 5 * d - e) / 6]
    assert p["beta"][0] == Fraction(13, 12) * (a - 2 * b + c) ** 2 + Fraction(1, 4) * (a - 4 * b + 3 * c) ** 2
    assert p["beta"][1] == Fraction(13, 12) * (b - 2 * c + d) ** 2 + Fraction(1, 4) * (b - d) ** 2
    assert p["beta"][2] == Fraction(13, 12) * (c - 2 * d + e) ** 2 + Fraction(1, 4) * (3 * c - 4 * d + e) ** 2
    f7 = [Fraction(x) for x in (2, 7, -1, 8, 2, -8, 1)]
    _, p = exact.weno_exact(f7, Fraction(1, 10 ** 6))
    a, b, c, d, e, f, g = f7
    assert p["d"] == [Fraction(1, 35), Fraction(12, 35), Fraction(18, 35), Fraction(4, 35)]
    assert p["q"][0] == (-3 * a + 13 * b - 23 * c + 25 * d) / 12
    assert p["q"][3] == (3 * d + 13 * e - 5 * f + g) / 12
    assert 240 * p["beta"][0] == (a * (547 * a - 3882 * b + 4642 * c - 1854 * d) + b * (7043 * b - 17246 * c + 7042 * d)
                                  + c * (11003 * c - 9402 * d) + 2107 * d * d)
    assert 240 * p["beta"][2] == (c * (547 * c - 2522 * d + 1922 * e - 494 * f) + d * (3443 * d - 5966 * e + 1602 * f)
                                  + e * (2843 * e - 1642 * f) + 267 * f * f)


@pytest.mark.parametrize("r", [3, 4])
def test_weno_linear_limit_and_constants(oracle, r):
    fn = oracle.weno5 if r == 3 else oracle.weno7
    lin = (np.array([2, -13, 47, 27, -3]) / 60.0 if r == 3
           else np.array([-3, 25, -101, 319, 214, -38, 4]) / 420.0)
    rng = np.random.default_rng(5)
    for _ in range(20):
        f = rng.uniform(-2, 2, size=2 * r - 1)
        assert abs(fn(f, 1e30) - lin @ f) < 1e-14        # eps -> inf: exactly the linear scheme
    assert fn(np.full(2 * r - 1, 1.7), 1e-6) == pytest.approx(1.7, abs=1e-15)
    # linear data f_j = j is reproduced exactly at j = 1/2 by every candidate
    j = np.arange(-r + 1, r, dtype=float)
    assert abs(fn(j, 1e-6) - 0.5) < 1e-14


@pytest.mark.parametrize("r,order", [(3, 5), (4, 7)])
def test_weno_measured_order_on_smooth_data(oracle, r, order):
    """Cell averages of sin over cells of width h -> point value of the primitive's derivative:
    the FD-WENO value at i+1/2 approximates h(x_{i+1/2}) where f_j = (1/h) int h; here we use the
    equivalent statement for cell averages of g: reconstruction of g at the face."""
    fn = oracle.weno5 if r == 3 else oracle.weno7
    errs = []
    hs = [0.2, 0.1, 0.05]
    for h in hs:
        x0 = 0.3
        j = np.arange(-r + 1, r)
        lo, hi = x0 + (j - 0.5) * h, x0 + (j + 0.5) * h
        avg = (-np.cos(hi) + np.cos(lo)) / h                  # cell averages of sin
        errs.append(abs(fn(avg, 1e-6 if r == 3 else 1e-2) - np.sin(x0 + 0.5 * h)))
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert min(orders) > order - 0.6, (errs, orders)


# ------------------------------------------------------------------ O5 LLF + WENO
@pytest.mark.parametrize("r", [3, 4])
def test_llf_flux_consistency(oracle, r):
    rng = np.random.default_rng(30)
    for _ in range(20):
        e, n = rng.uniform(0.2, 5), rng.uniform(0.1, 2)
        v = rng.uniform(-0.5, 0.5, 3)
        u = prim_to_cons(e, n, v)
        cells = np.tile(u, (2 * r, 1))
        for d in range(3):
            fh = oracle.llf_weno_flux(r, cells, d)
            assert np.max(np.abs(fh - flux_from_prim(e, n, v, d))) < 1e-14 * np.max(np.abs(u)) * 4


@pytest.mark.parametrize("r", [3, 4])
def test_llf_flux_scalar_advection_closed_form(oracle, r):
    """Uniform E, M (so v, p, alpha uniform); R varies.  The R flux is then the textbook scalar
    Lax-Friedrichs-split WENO flux for advection speed v_d: with eps -> inf it is the linear
    upwind-biased formula applied to f+ = (v+alpha)R/2 and mirrored to f- = (v-alpha)R/2."""
    lin = (np.array([2, -13, 47, 27, -3]) / 60.0 if r == 3
           else np.array([-3, 25, -101, 319, 214, -38, 4]) / 420.0)
    rng = np.random.default_rng(31)
    e, v = 1.3, np.array([0.3, -0.2, 0.1])
    cs = np.sqrt(1 / 3)
    for d in range(3):
        R = rng.uniform(0.5, 1.5, size=2 * r)
        cells = np.array([prim_to_cons(e, 1.0, v) for _ in range(2 * r)])
        cells[:, 4] = R
        v2 = v @ v
        alpha = (abs(v[d]) * (1 - 1 / 3) + cs * np.sqrt((1 - v2) * (1 - v[d] ** 2 - (v2 - v[d] ** 2) / 3))) / (1 - v2 / 3)
        fp = 0.5 * (v[d] + alpha) * R
        fm = 0.5 * (v[d] - alpha) * R
        expect = lin @ fp[:2 * r - 1] + lin @ fm[::-1][:2 * r - 1]
        got = oracle.llf_weno_flux(r, cells, d, eps=1e30)
        assert abs(got[4] - expect) < 1e-14
        # and the E, M components stay the exact physical flux
        assert np.max(np.abs(got[:4] - flux_from_prim(e, 1.0, v, d)[:4])) < 1e-14


@pytest.mark.parametrize("r", [3, 4])
def test_llf_alpha_is_max_over_all_2r_cells(oracle, r):
    """Q3: alpha is the max of a_d over the 2r cells i-r+1..i+r, including both end cells.  One fast
    cell (velocity along d only, so a_d = (|v|+cs)/(1+|v|cs)) is moved through every position; in the
    linear limit (eps -> inf) all five flux components have a closed form."""
    lin = (np.array([2, -13, 47, 27, -3]) / 60.0 if r == 3
           else np.array([-3, 25, -101, 319, 214, -38, 4]) / 420.0)
    cs = np.sqrt(1 / 3)
    m = 2 * r
    for d in range(3):
        for pos in range(m):
            prims = [(1.0 + 0.1 * k, 1.0 - 0.05 * k, np.zeros(3)) for k in range(m)]
            vf = np.zeros(3)
            vf[d] = -0.7
            prims[pos] = (prims[pos][0], prims[pos][1], vf)
            cells = np.array([prim_to_cons(*w) for w in prims])
            F = np.array([flux_from_prim(*w, d) for w in prims])
            alpha = (0.7 + cs) / (1 + 0.7 * cs)          # > cs of the cells at rest
            fp = 0.5 * (F + alpha * cells)
            fm = 0.5 * (F - alpha * cells)
            expect = lin @ fp[:m - 1] + lin @ fm[::-1][:m - 1]
            got = oracle.llf_weno_flux(r, cells, d, eps=1e30)
            assert np.max(np.abs(got - expect)) < 1e-13, (d, pos)


# ------------------------------------------------------------------ O7 MUSTA-FORCE
def test_musta_consistency(oracle):
    rng = np.random.default_rng(40)
    for _ in range(20):
        e, n = rng.uniform(0.2, 5), rng.uniform(0.1, 2)
        v = rng.uniform(-0.5, 0.5, 3)
        u = prim_to_cons(e, n, v)
        cells = np.tile(u, (4, 1))
        for d in range(3):
            for K in (1, 2, 3):
                fs = oracle.musta_force_flux(cells, d, K=K)
                assert np.max(np.abs(fs - flux_from_prim(e, n, v, d))) < 4e-14 * np.max(np.abs(u))


def _scalar_musta(RL, RR, v, tau, K):
    """K-stage FORCE recursion for the scalar flux f = v R with fixed tau."""
    for stage in range(1, K + 1):
        FL, FR = v * RL, v * RR
        RM = 0.5 * (RL + RR) - 0.5 * tau * (FR - FL)
        FM = v * RM
        F = 0.25 * (FL + 2 * FM + FR - (RR - RL) / tau)
        if stage == K:
            return F
        RL, RR = RL - tau * (F - FL), RR - tau * (FR - F)


@pytest.mark.parametrize("K", [1, 2, 3])
def test_musta_scalar_closed_form(oracle, K):
    """Uniform E, M; R piecewise: minmod slopes vanish if R is a step with flat neighbours, so
    Q_L = u_i, Q_R = u_{i+1}.  E, M fluxes are exact and correctors leave E, M unchanged, so tau is
    the same in every stage and the R flux follows the scalar recursion; K=1 has the closed form
    F = v(R_L+R_R)/2 - (tau v^2 + 1/tau)(R_R-R_L)/4."""
    e, v = 2.0, np.array([0.25, -0.1, 0.3])
    cs = np.sqrt(1 / 3)
    for d in range(3):
        cells = np.array([prim_to_cons(e, 1.0, v) for _ in range(4)])
        RL, RR = 1.2, 0.7
        cells[:2, 4], cells[2:, 4] = RL, RR
        v2 = v @ v
        S = (abs(v[d]) * (2 / 3) + cs * np.sqrt((1 - v2) * (1 - v[d] ** 2 - (v2 - v[d] ** 2) / 3))) / (1 - v2 / 3)
        tau = 0.9 / S
        got = oracle.musta_force_flux(cells, d, K=K, C=0.9)
        assert abs(got[4] - _scalar_musta(RL, RR, v[d], tau, K)) < 1e-14
        if K == 1:
            closed = 0.5 * v[d] * (RL + RR) - 0.25 * (tau * v[d] ** 2 + 1 / tau) * (RR - RL)
            assert abs(got[4] - closed) < 1e-14
        assert np.max(np.abs(got[:4] - flux_from_prim(e, 1.0, v, d)[:4])) < 1e-13


def test_musta_muscl_face_states(oracle):
    """O6: Q_L = u_i + minmod/2, Q_R = u_{i+1} - minmod/2 on the R component (E, M uniform)."""
    e, v = 2.0, np.array([0.25, 0.0, 0.0])
    cells = np.array([prim_to_cons(e, 1.0, v) for _ in range(4)])
    R = np.array([1.0, 1.2, 1.5, 1.6])
    cells[:, 4] = R
    QL = R[1] + 0.5 * min(R[1] - R[0], R[2] - R[1])
    QR = R[2] - 0.5 * min(R[2] - R[1], R[3] - R[2])
    cs = np.sqrt(1 / 3)
    tau = 0.9 / ((0.25 + cs) / (1 + 0.25 * cs))
    got = oracle.musta_force_flux(cells, 0, K=2)
    assert abs(got[4] - _scalar_musta(QL, QR, 0.25, tau, 2)) < 1e-14
    # a local extremum kills the slope
    R2 = np.array([1.0, 1.4, 1.2, 1.3])
    cells[:, 4] = R2
    got = oracle.musta_force_flux(cells, 0, K=1)
    assert abs(got[4] - _scalar_musta(R2[1], R2[2], 0.25, tau, 1)) < 1e-14
