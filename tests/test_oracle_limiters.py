"""Pins of the oracle's slope limiters (O6', "a variety of slope limiting methods").
Nothing here retypes the oracle's formulas: the expected values are textbook numbers and the defining
properties (Sweby's second-order TVD region in the flux-limiter form phi(r), r = b/a)."""
import itertools
import math

import numpy as np
import pytest

from paper_1604_03360_b200 import workloads as W

LIMS = [0, 1, 2, 3]
NAMES = {0: "minmod", 1: "vanleer", 2: "mc", 3: "superbee"}


def test_textbook_values(oracle):
    # (a, b) = (1, 3):  minmod 1, van Leer 2*3/4, MC min(2, 6, 2), superbee max(min(2,3), min(1,6))
    assert [oracle.limited_slope(l, 1.0, 3.0) for l in LIMS] == [1.0, 1.5, 2.0, 2.0]
    # (1, 1.5): minmod 1, van Leer 3/2.5, MC min(2, 3, 1.25), superbee max(min(2,1.5), min(1,3))
    got = [oracle.limited_slope(l, 1.0, 1.5) for l in LIMS]
    assert got[0] == 1.0 and abs(got[1] - 1.2) < 1e-15 and got[2] == 1.25 and got[3] == 1.5


@pytest.mark.parametrize("lim", LIMS)
def test_defining_properties(oracle, lim):
    rng = np.random.default_rng(28)
    for _ in range(400):
        a, b = rng.normal(size=2) * 10.0 ** rng.integers(-3, 3)
        s = oracle.limited_slope(lim, a, b)
        assert s == oracle.limited_slope(lim, b, a) or abs(s - oracle.limited_slope(lim, b, a)) <= 1e-15 * abs(s)
        assert abs(oracle.limited_slope(lim, -a, -b) + s) <= 1e-15 * abs(s)               # odd
        assert abs(oracle.limited_slope(lim, 3.0 * a, 3.0 * b) - 3.0 * s) <= 1e-14 * abs(s)  # homogeneous
        if a * b <= 0.0:
            assert s == 0.0                                                              # extremum: flat
        else:
            assert s * a > 0.0
            assert abs(s) <= 2.0 * min(abs(a), abs(b)) * (1 + 1e-15)                      # TVD bound
            assert abs(s) >= min(abs(a), abs(b)) * (1 - 1e-15)                            # at least minmod
            assert abs(s) <= max(abs(a), abs(b)) * (1 + 1e-15)
    for v in (0.3, -7.0):
        assert abs(oracle.limited_slope(lim, v, v) - v) <= 1e-15 * abs(v)                # a = b: the slope itself


def test_ordering_minmod_le_vanleer_le_superbee(oracle):
    """In the TVD region minmod is the lower and superbee the upper boundary; van Leer and MC lie between."""
    for a, b in itertools.product([0.2, 1.0, 2.5, 9.0], repeat=2):
        mm, vl, mc, sb = [oracle.limited_slope(l, a, b) for l in LIMS]
        assert mm <= vl + 1e-15 and mm <= mc + 1e-15 and vl <= sb + 1e-15 and mc <= sb + 1e-15


@pytest.mark.parametrize("lim", [1, 2, 3])
def test_face_states_use_the_limiter(oracle, lim):
    """Uniform E, M (at rest, so the E and M fluxes and correctors are exact): the K = 1 MUSTA-FORCE flux of R
    has the closed form of the scalar FORCE flux at speed 0, F_R = -(1/(4 tau)) (Q_R - Q_L), with the MUSCL
    face states built from the limited slopes."""
    e = 1.5
    R = np.array([1.0, 2.0, 5.0, 6.5])
    cells = np.zeros((4, 5))
    cells[:, 0] = e
    cells[:, 4] = R
    sl1 = oracle.limited_slope(lim, R[1] - R[0], R[2] - R[1])
    sl2 = oracle.limited_slope(lim, R[2] - R[1], R[3] - R[2])
    QL, QR = R[1] + 0.5 * sl1, R[2] - 0.5 * sl2
    tau = 0.9 / math.sqrt(1.0 / 3.0)                     # S = c_s at rest
    got = oracle.musta_force_flux(cells, 0, K=1, C=0.9, limiter=lim)
    assert abs(got[4] - (-(QR - QL) / (4.0 * tau))) < 1e-14
    assert abs(got[4] - oracle.musta_force_flux(cells, 0, K=1, C=0.9, limiter=0)[4]) > 1e-3   # not minmod's


@pytest.mark.parametrize("lim", LIMS)
def test_second_order_on_smooth_data(oracle, lim):
    """Charge advection (uniform e, v; smooth periodic n): L1 error of R falls with order about 2 for every
    limiter (clipping at extrema costs a little)."""
    errs = []
    for n in (32, 64, 128):
        dx = 1.0 / n
        x = W.cell_centres(n, dx, 0.0)
        e, v = 1.0, 0.4
        nn = 1.0 + 0.3 * np.sin(2 * np.pi * x)
        z = np.zeros(n)
        cons = W.prim_to_cons(np.full(n, e), nn, np.full(n, v), z, z).reshape(5, 1, 1, n)
        o = oracle.Oracle(n, 1, 1, dx, W.MUSTA_FORCE, bc_x=W.BC_PERIODIC, limiter=lim)
        o.set_state(cons)
        T, steps = 0.25, int(round(0.25 / (0.2 * dx)))
        o.step(T / steps, steps)
        u = o.get_state()[4, 0, 0]
        g = 1.0 / math.sqrt(1 - v * v)
        exact = (1.0 + 0.3 * np.sin(2 * np.pi * (x - v * T))) * g
        errs.append(np.sum(np.abs(u - exact)) * dx)
    order = math.log2(errs[0] / errs[2]) / 2
    assert 1.5 < order < 2.6, (NAMES[lim], errs, order)
