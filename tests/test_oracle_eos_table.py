"""Pins of the oracle's tabulated closure p(e) (SURVEY 8(f)-N1 second half; PAPER.md:7 motivates a general equation
of state).  CPU only.  Expected values come from the definitions: the conserved variables of a state with pressure
numpy.interp(e, grid, table) (a library routine, not the oracle's lookup), the closed-form p = e/3 path, the
spectrum of a numerically differentiated flux, and exact conservation."""
import math

import numpy as np
import pytest

from paper_1604_03360_b200 import workloads as W


def cons_with_pressure(e, p, n, v):
    """Definition of the conserved variables for a given pressure (no equation of state inside)."""
    v = np.asarray(v, dtype=float)
    g2 = 1.0 / (1.0 - v @ v)
    w = (e + p) * g2
    return np.array([w - p, w * v[0], w * v[1], w * v[2], n * math.sqrt(g2)])


def test_a_linear_table_is_the_closed_form_gas(oracle):
    """p = e/3 sampled on any grid is reproduced exactly by linear interpolation: the iterative con2prim and the
    general speed formula must then give what the closed-form p = e/3 path gives."""
    rng = np.random.default_rng(5)
    tab = np.linspace(0.0, 50.0, 77) / 3.0
    for _ in range(200):
        e = rng.uniform(0.05, 45.0)
        sp = rng.uniform(0.0, 0.95)
        d = rng.standard_normal(3)
        v = sp * d / np.linalg.norm(d)
        u = cons_with_pressure(e, e / 3.0, rng.uniform(0.1, 2.0), v)
        prim, speeds, flag = oracle.con2prim_table(u, tab, 0.0, 50.0)
        ref, flag0 = oracle.con2prim(u)
        assert flag == 0 and flag0 == 0
        assert np.allclose(prim[:6], ref, rtol=2e-13 / (1 - sp * sp), atol=0)
        assert abs(prim[6] - 1.0 / 3.0) < 1e-14
        for ax in range(3):
            assert abs(speeds[ax] - oracle.signal_speed(ref[3:6], ax)) <= 1e-13 / (1 - sp * sp)


@pytest.mark.parametrize("n_tab", [64, 1000, 4096])
def test_round_trip_through_a_nonlinear_table(oracle, n_tab):
    """prim -> cons with the pressure numpy.interp gives -> the oracle's con2prim must return the state: pins the
    Newton iteration, the segment index (an off-by-one breaks it) and the continuation beyond the table's end."""
    tab, e0, e1 = W.crossover_eos_table(n=n_tab, e_max=30.0)
    grid = np.linspace(e0, e1, n_tab)
    rng = np.random.default_rng(11)
    for trial in range(300):
        e = rng.uniform(0.02, 29.5) if trial % 10 else rng.uniform(30.5, 40.0)     # some beyond the last node
        if e <= e1:
            p = float(np.interp(e, grid, tab))
        else:                                                                      # continued last segment
            p = tab[-1] + (e - grid[-1]) * (tab[-1] - tab[-2]) / (grid[-1] - grid[-2])
        sp = rng.uniform(0.0, 0.9)
        d = rng.standard_normal(3)
        v = sp * d / np.linalg.norm(d)
        nn = rng.uniform(0.1, 2.0)
        u = cons_with_pressure(e, p, nn, v)
        prim, speeds, flag = oracle.con2prim_table(u, tab, e0, e1)
        assert flag == 0
        tol = 1e-12 / (1 - sp * sp)
        assert abs(prim[0] - e) <= tol * e and abs(prim[1] - p) <= tol * max(p, e)
        assert abs(prim[2] - nn) <= tol * nn
        assert np.max(np.abs(prim[3:6] - v)) <= tol
        i = min(max(int(math.floor((e - e0) / (grid[1] - grid[0]))), 0), n_tab - 2)
        assert abs(prim[6] - (tab[i + 1] - tab[i]) / (grid[1] - grid[0])) <= 1e-12


def test_speeds_are_the_spectrum_of_the_flux_jacobian(oracle):
    """a_d = max |eigenvalue| of dF_d/dU, F_d evaluated through the oracle's own con2prim with the table, the
    derivative by central differences inside one table segment (where p(e) is smooth)."""
    tab, e0, e1 = W.crossover_eos_table(n=40, e_max=20.0)        # wide segments: the stencil stays inside one
    grid = np.linspace(e0, e1, 40)
    rng = np.random.default_rng(3)

    def flux(u, d):
        prim, _, _ = oracle.con2prim_table(u, tab, e0, e1)
        p, v = prim[1], prim[3:6]
        F = np.array([u[1 + d], u[1] * v[d], u[2] * v[d], u[3] * v[d], u[4] * v[d]])
        F[1 + d] += p
        return F

    for _ in range(25):
        k = rng.integers(2, 38)
        e = grid[k] + 0.5 * (grid[1] - grid[0])                  # middle of a segment
        p = float(np.interp(e, grid, tab))
        sp = rng.uniform(0.05, 0.8)
        dvec = rng.standard_normal(3)
        v = sp * dvec / np.linalg.norm(dvec)
        u = cons_with_pressure(e, p, 0.7, v)
        _, speeds, _ = oracle.con2prim_table(u, tab, e0, e1)
        for d in range(3):
            J = np.zeros((5, 5))
            for c in range(5):
                h = 1e-6 * max(abs(u[c]), abs(u[0]))
                up, um = u.copy(), u.copy()
                up[c] += h
                um[c] -= h
                J[:, c] = (flux(up, d) - flux(um, d)) / (2 * h)
            lam = np.linalg.eigvals(J)
            assert np.max(np.abs(lam.imag)) < 1e-5
            assert abs(np.max(np.abs(lam.real)) - speeds[d]) < 2e-6
            assert speeds[d] < 1.0


@pytest.mark.parametrize("scheme", [W.WENO5, W.WENO7, W.MUSTA_FORCE])
def test_whole_solver_with_a_table(oracle, scheme):
    """(a) with the linear p = e/3 table the solver must reproduce the closed-form solver's L(u) and steps; (b) with
    the crossover table it conserves E, M, R on a periodic grid, keeps a uniform state, and differs from the gas."""
    n = (20, 12, 9)
    big = W.lumpy(n=max(n), hotspots=12, with_velocity=True, scheme=scheme, box=max(n) / 16.0, sigma_unit=0.12)
    cons = np.ascontiguousarray(big.cons[:, :n[2], :n[1], :n[0]])
    w0 = W.Workload("gas", n, big.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, cons, 0.0, cfl=0.2, nsteps=5)
    wl = W.Workload("lin", n, big.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, cons, 0.0, cfl=0.2, nsteps=5,
                    eos_table=(np.linspace(0.0, 60.0, 301) / 3.0, 0.0, 60.0))
    o0, ol = oracle.from_workload(w0), oracle.from_workload(wl)
    L0, Ll = o0.eval_L(cons), ol.eval_L(cons)
    scale = np.max(np.abs(cons[0])) / w0.dx
    assert np.max(np.abs(L0 - Ll)) <= 1e-12 * scale
    oracle.run(o0, w0)
    oracle.run(ol, wl)
    assert np.max(np.abs(o0.get_state() - ol.get_state())) <= 1e-12 * np.max(np.abs(cons[0]))

    wc = W.Workload("xover", n, big.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, cons, 0.0, cfl=0.2, nsteps=10,
                    eos_table=W.crossover_eos_table(n=512, e_max=60.0))
    oc = oracle.from_workload(wc)
    assert np.max(np.abs(oc.eval_L(cons) - L0)) > 1e-3 * scale           # it is another operator
    tot0 = [math.fsum(cons[c].ravel()) for c in range(5)]
    oracle.run(oc, wc)
    u = oc.get_state()
    for c in range(5):
        assert abs(math.fsum(u[c].ravel()) - tot0[c]) <= 1e-13 * tot0[0] * 10
    # uniform state
    u0 = cons_with_pressure(1.7, float(np.interp(1.7, np.linspace(0, 60.0, 512), wc.eos_table[0])), 0.3,
                            [0.31, -0.22, 0.13])
    uni = np.broadcast_to(u0.reshape(5, 1, 1, 1), (5, n[2], n[1], n[0])).copy()
    wu = W.Workload("uni", n, big.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, uni, 0.0, eos_table=wc.eos_table)
    ou = oracle.from_workload(wu)
    assert np.all(ou.eval_L(uni) == 0.0)
