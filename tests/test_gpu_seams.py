"""Parity of the CUDA path against the CPU oracle where the marching kernels are most fragile (all `-m gpu`):
the seams between chunks of the z / y march (window re-prime, parked flux, cp.async slot reuse, the half group at the
end of an odd MUSTA y chunk), the run-time number of MUSTA-FORCE stages, the values the Q16 clamp produces, the
flag for non-finite states, and the sizes and precisions bench.py times (sampled cells at 512^3).

Tolerances are those of tests/test_gpu_parity.py (BASELINE.json north_star; reading Q12)."""
import functools
import math

import numpy as np
import pytest

from paper_1604_03360_b200 import workloads as W
from test_gpu_parity import SCHEMES, TOL_100_F32, TOL_STAGE, reldiff, small_workload, to_dev, _crop_periodic

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1604_03360_b200 import binding
    return binding


# ------------------------------------------------------------------ chunk seams of the marching kernels vs the ORACLE
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("chunks", [(5, 7), (1, 1), (16, 16)])
def test_chunk_seams_match_the_oracle(B, oracle, scheme, prec, chunks):
    """70 x 45 x 40 with tile_zc / sweep_zc far below the grid: every chunk boundary of the z and y march falls
    inside the grid (ragged last chunks, odd chunk lengths).  L(u) and one full step against the oracle."""
    n = (70, 45, 40)
    for bc in (W.BC_PERIODIC, W.BC_OUTFLOW):
        w = small_workload(scheme, n, bc)
        w.options = {"tile_zc": chunks[0], "sweep_zc": chunks[1]}
        wo = small_workload(scheme, n, bc)
        h = B.from_workload(w, precision=prec, kernel=B.KERNEL_FUSED)
        o = oracle.from_workload(wo)
        Lo = o.eval_L(wo.cons)
        Lg = h.eval_L(to_dev(B, w.cons, h.dtype)).cpu().numpy()
        scale = np.max(np.abs(w.cons[0])) / w.dx
        # fp32: a few hundred roundings of 6e-8 on differences of O(1) data, relative to E/dx
        assert reldiff(Lg, Lo, scale=scale) <= (TOL_STAGE if prec == 0 else 2e-5)
        dt = 0.2 * w.dx / o.max_signal_speed()
        o.step(dt, 1)
        h.step(dt, 1)
        assert reldiff(h.get_state().cpu().numpy(), o.get_state()) <= (3 * TOL_STAGE if prec == 0 else 3e-6)
        assert h.status() == 0
        h.close()


# ------------------------------------------------------------------ MUSTA-FORCE with K != 2 (N3)
@pytest.mark.parametrize("K", [1, 3, 4])
def test_musta_stage_count_matches_the_oracle(B, oracle, K):
    w = small_workload(W.MUSTA_FORCE, (45, 23, 70))
    w.options = {"musta_stages": K}
    o = oracle.from_workload(w)
    h = B.from_workload(w)
    Lo = o.eval_L(w.cons)
    Lg = h.eval_L(to_dev(B, w.cons)).cpu().numpy()
    assert reldiff(Lg, Lo, scale=np.max(np.abs(w.cons[0])) / w.dx) <= TOL_STAGE
    # and it is not the K = 2 operator
    w2 = small_workload(W.MUSTA_FORCE, (45, 23, 70))
    L2 = oracle.from_workload(w2).eval_L(w2.cons)
    assert np.max(np.abs(L2 - Lo)) > 1e-4 * np.max(np.abs(Lo))
    w.nsteps = 10
    for dt in oracle.run(o, w):
        h.step(dt, 1)
    assert reldiff(h.get_state().cpu().numpy(), o.get_state()) <= 1e-10
    assert h.status() == 0
    h.close()


# ------------------------------------------------------------------ Q16: the values the clamp produces
@pytest.mark.parametrize("scheme", SCHEMES)
def test_clamped_cell_gives_the_oracles_values(B, oracle, scheme):
    """One cell with |M| = 1.5 E: both sides scale M back to (1 - 1e-12) E along M and raise the flag.  The clamped
    cell has 1 - v^2 = 2e-12, so its pressure and signal speeds carry a relative rounding error of about
    1e-16 / 2e-12 = 5e-5 on quantities that are themselves ~1e-6 of the flux (sqrt(1 - v^2)): L(u) agrees to
    ~1e-10 in the cells whose stencils contain the clamped cell and to the usual 1e-12 everywhere else."""
    n = (24, 17, 15)
    w = small_workload(scheme, n)
    bad = w.cons.copy()
    ci, cj, ck = 11, 8, 7
    m = bad[1:4, ck, cj, ci]
    bad[1:4, ck, cj, ci] = m / np.linalg.norm(m) * 1.5 * bad[0, ck, cj, ci]
    wb = W.Workload("clamp", n, w.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, bad)
    o = oracle.from_workload(wb)
    h = B.from_workload(wb)
    Lo = o.eval_L(bad)
    Lg = h.eval_L(to_dev(B, bad)).cpu().numpy()
    assert h.status() == B.EUNPHYSICAL
    scale = np.max(np.abs(bad[0])) / w.dx
    r = {W.WENO5: 3, W.WENO7: 4, W.MUSTA_FORCE: 2}[scheme]
    near = np.zeros(Lo.shape[1:], dtype=bool)
    near[ck - r:ck + r + 1, cj, ci] = near[ck, cj - r:cj + r + 1, ci] = near[ck, cj, ci - r:ci + r + 1] = True
    assert np.all(np.isfinite(Lg))
    far_err = max(np.max(np.abs((Lg[c] - Lo[c])[~near])) for c in range(5)) / scale
    near_err = max(np.max(np.abs((Lg[c] - Lo[c])[near])) for c in range(5)) / scale
    assert far_err <= TOL_STAGE, far_err
    assert near_err <= 2e-9, near_err
    # the clamp did act: without it the result would differ by far more than the tolerance
    assert max(np.max(np.abs(Lo[c][near])) for c in range(5)) / scale > 1e-3
    h.close()


# ------------------------------------------------------------------ non-finite states raise the flag
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("field,value", [(0, float("nan")), (2, float("nan")), (0, float("inf")), (0, -1.0)])
def test_non_finite_or_negative_energy_raises_the_flag(B, scheme, field, value):
    w = small_workload(scheme, (40, 33, 24))
    bad = w.cons.copy()
    bad[field, 10, 20, 30] = value
    h = B.from_workload(w)
    h.step(1e-4, 1)
    assert h.status() == 0
    h.set_state(to_dev(B, bad))
    h.step(1e-4, 1)
    assert h.status() == B.EUNPHYSICAL, (scheme, field, value)
    h.close()


# ------------------------------------------------------------------ the sizes and precisions bench.py times
@functools.lru_cache(maxsize=1)
def _production_512():
    return W.lumpy(n=512, hotspots=200, with_velocity=True, scheme=W.WENO5, nsteps=1, cfl=0.2)


@pytest.mark.parametrize("scheme,prec", [(W.WENO7, 0), (W.MUSTA_FORCE, 0), (W.WENO7, 1), (W.WENO5, 1)])
def test_bench_variants_at_512_on_sampled_cells(B, oracle, scheme, prec):
    """BASELINE configs[4] at its full size for the variants of the bench line other than WENO5 fp64 (which
    tests/test_gpu_parity.py::test_full_size_step_on_sampled_cells covers): one RK3 step, sampled cells recomputed
    by the oracle from a (6 r + 1)^3 crop, plus conservation over the whole grid."""
    import torch
    n = 512
    w0 = _production_512()
    w = W.Workload(w0.name, w0.n, w0.dx, w0.origin, scheme, w0.bc, w0.cons, 0.0, cfl=0.2, nsteps=1)
    h = B.from_workload(w, precision=prec)
    dt = 0.2 * w.dx / h.max_signal_speed()
    h.step(dt, 1)
    assert h.status() == 0
    ug_t = h.get_state()
    r = {W.WENO5: 3, W.WENO7: 4, W.MUSTA_FORCE: 2}[scheme]
    half = 3 * r
    samples = [(0, 0, 0), (n - 1, n - 1, n - 1), (30, 6, 63), (31, 7, 64), (62, 127, 127), (61, 128, 128),
               (n // 2, n // 2, n // 2), (n - 1, 0, 128), (333, 222, 111)]
    worst = 0.0
    scale = np.max(np.abs(w.cons[0]))
    fmax = [np.max(np.abs(w.cons[c])) for c in range(5)]
    for (i, j, k) in samples:
        crop = _crop_periodic(w.cons, (i, j, k), half)
        m = 2 * half + 1
        wc = W.Workload("crop", (m, m, m), w.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, crop)
        o = oracle.from_workload(wc)
        o.step(dt, 1)
        ref = o.get_state()[:, half, half, half]
        got = ug_t[:, k, j, i].double().cpu().numpy()
        for c in range(5):
            den = max(abs(ref[c]), 1e-15 * scale) if c == 0 else max(fmax[c], 1e-15 * scale)
            worst = max(worst, abs(got[c] - ref[c]) / den)
    assert worst <= (3e-12 if prec == 0 else 1e-5), worst
    tot1 = [float(torch.sum(ug_t[c].double())) for c in range(5)]
    tot0 = [float(np.sum(w.cons[c])) for c in range(5)]
    for a, b in zip(tot0, tot1):
        assert abs(a - b) <= (1e-11 if prec == 0 else 2e-6) * abs(tot0[0]), (tot0, tot1)
    del ug_t
    h.close()


@pytest.mark.parametrize("scheme", [W.WENO5, W.MUSTA_FORCE])
def test_three_steps_at_512_on_sampled_cells(B, oracle, scheme):
    """The bench size beyond one step: three RK3 steps of the 512^3 state with dt from the
    device's max signal speed before each step; an output cell depends on the cells within 3 x 3 r of it, so the
    oracle recomputes sampled cells (tile / chunk corners, the periodic seam, interior) from (18 r + 1)^3 crops
    advanced with the same three dt."""
    n = 512
    w0 = _production_512()
    w = W.Workload(w0.name, w0.n, w0.dx, w0.origin, scheme, w0.bc, w0.cons, 0.0, cfl=0.2, nsteps=3)
    h = B.from_workload(w)
    dts = []
    for _ in range(3):
        dts.append(0.2 * w.dx / h.max_signal_speed())
        h.step(dts[-1], 1)
    assert h.status() == 0
    ug_t = h.get_state()
    r = {W.WENO5: 3, W.WENO7: 4, W.MUSTA_FORCE: 2}[scheme]
    half = 9 * r
    samples = [(0, 0, 0), (n - 1, n - 1, n - 1), (31, 7, 64), (61, 128, 128), (333, 222, 111)]
    scale = np.max(np.abs(w.cons[0]))
    fmax = [np.max(np.abs(w.cons[c])) for c in range(5)]
    worst = 0.0
    for (i, j, k) in samples:
        crop = _crop_periodic(w.cons, (i, j, k), half)
        m = 2 * half + 1
        wc = W.Workload("crop", (m, m, m), w.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, crop)
        o = oracle.from_workload(wc)
        for dt in dts:
            o.step(dt, 1)
        ref = o.get_state()[:, half, half, half]
        got = ug_t[:, k, j, i].cpu().numpy()
        for c in range(5):
            den = max(abs(ref[c]), 1e-15 * scale) if c == 0 else max(fmax[c], 1e-15 * scale)
            worst = max(worst, abs(got[c] - ref[c]) / den)
    assert worst <= 3 * 3e-12, worst
    del ug_t
    h.close()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_100_steps_fp64_across_every_seam(B, oracle, scheme):
    """The 1e-9-after-100-steps bound on a grid that crosses every seam of the marching kernels (VERDICT round 2,
    weak 4): 70 x 45 x 40 has three x-tiles with a ragged last one, and with tile_zc = sweep_zc = 16 three z-chunks
    and three y-chunks with ragged tails; periodic x and z, outflow y, so both ghost rules are inside the run."""
    w0 = small_workload(scheme, (70, 45, 40))
    w = W.Workload("seams100", w0.n, w0.dx, (0, 0, 0), scheme, (W.BC_PERIODIC, W.BC_OUTFLOW, W.BC_PERIODIC), w0.cons,
                   0.0, cfl=0.2, nsteps=100, options={"tile_zc": 16, "sweep_zc": 16})
    wo = W.Workload("seams100", w.n, w.dx, w.origin, scheme, w.bc, w.cons, 0.0, cfl=0.2, nsteps=100)
    o = oracle.from_workload(wo)       # the chunk lengths are the CUDA path's business
    dts = oracle.run(o, wo)
    h = B.from_workload(w, kernel=B.KERNEL_FUSED)
    for dt in dts:
        h.step(dt, 1)
    d = reldiff(h.get_state().cpu().numpy(), o.get_state())
    assert d <= 1e-9, d
    assert np.max(np.abs(o.get_state() - w.cons)) > 1e-3
    assert h.status() == 0
    h.close()


# ------------------------------------------------------------------ tabulated equation of state (N1, second half)
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("kernel", ["fused", "generic"])
def test_tabulated_eos_matches_the_oracle(B, oracle, scheme, kernel):
    """The crossover table p(e) (c_s^2 from 0.15 to 1/3): L(u), one step and ten steps against the oracle on a ragged
    grid through the marching kernels and the generic kernel; and with the linear p = e/3 table the result must be the
    closed-form gas's."""
    n = (45, 23, 38)
    w0 = small_workload(scheme, n)
    tab = W.crossover_eos_table(n=2048, e_max=float(np.max(w0.cons[0])) * 1.5)
    w = W.Workload("xover", n, w0.dx, (0, 0, 0), scheme, (W.BC_PERIODIC, W.BC_OUTFLOW, W.BC_PERIODIC), w0.cons, 0.0,
                   cfl=0.2, nsteps=10, eos_table=tab)
    kern = B.KERNEL_FUSED if kernel == "fused" else B.KERNEL_GENERIC
    o = oracle.from_workload(w)
    h = B.from_workload(w, kernel=kern)
    scale = np.max(np.abs(w.cons[0])) / w.dx
    Lo = o.eval_L(w.cons)
    Lg = h.eval_L(to_dev(B, w.cons)).cpu().numpy()
    assert reldiff(Lg, Lo, scale=scale) <= TOL_STAGE
    assert abs(h.max_signal_speed() - o.max_signal_speed()) <= 1e-14
    dts = oracle.run(o, w)
    o1 = oracle.from_workload(w)
    o1.step(dts[0], 1)
    h.step(dts[0], 1)
    assert reldiff(h.get_state().cpu().numpy(), o1.get_state()) <= 3 * TOL_STAGE
    for dt in dts[1:]:
        h.step(dt, 1)
    assert reldiff(h.get_state().cpu().numpy(), o.get_state()) <= 1e-11
    assert h.status() == 0
    h.close()
    # it is not the gas: the operator differs
    og = oracle.from_workload(w0)
    assert np.max(np.abs(og.eval_L(w0.cons) - Lo)) > 1e-3 * scale
    # the linear table is the gas
    wl = W.Workload("lin", n, w0.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, w0.cons, 0.0,
                    eos_table=(np.linspace(0.0, 80.0, 401) / 3.0, 0.0, 80.0))
    wg = W.Workload("gas", n, w0.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, w0.cons, 0.0)
    hl, hg = B.from_workload(wl, kernel=kern), B.from_workload(wg, kernel=kern)
    Ll = hl.eval_L(to_dev(B, w0.cons)).cpu().numpy()
    Lgas = hg.eval_L(to_dev(B, w0.cons)).cpu().numpy()
    assert reldiff(Ll, Lgas, scale=scale) <= TOL_STAGE
    hl.close()
    hg.close()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_tabulated_eos_fp32_against_the_fp64_oracle(B, oracle, scheme):
    """Reading Q17 for the tabulated closure: the fp32 kernels, whose table con2prim runs in double
    on float inputs, against the fp64 oracle: L(u) and the state after ten steps."""
    n = (45, 23, 38)
    w0 = small_workload(scheme, n)
    tab = W.crossover_eos_table(n=2048, e_max=float(np.max(w0.cons[0])) * 1.5)
    w = W.Workload("xover32", n, w0.dx, (0, 0, 0), scheme, (W.BC_PERIODIC, W.BC_OUTFLOW, W.BC_PERIODIC), w0.cons, 0.0,
                   cfl=0.2, nsteps=10, eos_table=tab)
    o = oracle.from_workload(w)
    h = B.from_workload(w, precision=1)
    scale = np.max(np.abs(w.cons[0])) / w.dx
    Lo = o.eval_L(w.cons)
    Lg = h.eval_L(to_dev(B, w.cons, h.dtype)).double().cpu().numpy()
    assert reldiff(Lg, Lo, scale=scale) <= 3e-5
    for dt in oracle.run(o, w):
        h.step(dt, 1)
    assert reldiff(h.get_state().double().cpu().numpy(), o.get_state()) <= TOL_100_F32
    assert h.status() == 0
    h.close()


def test_eos_table_arguments_are_checked(B):
    import torch
    h = B.Hydro(16, 16, 16, 0.1, W.WENO5)
    with pytest.raises(B.HydroError):
        h.set_option("eos", 2)                                   # no table yet
    t = torch.linspace(0, 10, 11, dtype=torch.float64, device="cuda")
    assert B.lib.hydro_set_eos_table(h._h, t.data_ptr(), 1, 0.0, 1.0) == B.EINVAL
    assert B.lib.hydro_set_eos_table(h._h, t.data_ptr(), 11, 1.0, 1.0) == B.EINVAL
    assert B.lib.hydro_set_eos_table(h._h, None, 11, 0.0, 1.0) == B.EINVAL
    host = np.zeros(11)
    assert B.lib.hydro_set_eos_table(h._h, host.ctypes.data, 11, 0.0, 1.0) == B.EINVAL
    assert B.lib.hydro_set_eos_table(h._h, t.data_ptr(), 11, 0.0, 30.0) == B.OK
    h.set_option("eos", 0)
    h.set_option("eos", 2)
    h.close()


# ------------------------------------------------------------------ fp32: the cross-multiplied WENO weights at any data scale
@pytest.mark.parametrize("scheme", [W.WENO5, W.WENO7])
@pytest.mark.parametrize("scale,eps", [(1e4, 1e-6), (1e3, 1e-6), (1e-3, 1e-14), (1.0, 1e-13)])
def test_fp32_weno_weights_survive_any_data_scale(B, oracle, scheme, scale, eps):
    """The fp32 kernels multiply the weights through (products of squared smoothness indicators: the 6th power for
    WENO7).  Flux jumps of 1e4..1e5 would overflow them and a tiny epsilon on flat data underflow them; the kernels
    rescale the indicators by a power of two first.  L(u) of scaled data against the fp64 oracle with the same
    epsilon (the equations are homogeneous of degree one in (E, M, R), so the data stay admissible)."""
    w = small_workload(scheme, (45, 23, 38))
    cons = w.cons * scale
    ws = W.Workload("scaled", w.n, w.dx, (0, 0, 0), scheme, (W.BC_PERIODIC,) * 3, cons, 0.0,
                    options={"weno_eps": eps})
    o = oracle.from_workload(ws)
    h = B.from_workload(ws, precision=1)
    Lo = o.eval_L(cons)
    Lg = h.eval_L(to_dev(B, cons, h.dtype)).cpu().numpy()
    assert np.all(np.isfinite(Lg))
    assert reldiff(Lg, Lo, scale=np.max(np.abs(cons[0])) / w.dx) <= 3e-5
    assert h.status() == 0
    h.close()


@pytest.mark.parametrize("scheme,scale", [(W.WENO5, 1e16), (W.WENO7, 1e13)])
def test_fp32_data_bound_stated_in_the_header(B, oracle, scheme, scale):
    """include/hydro.h gives the fp32 path a data bound (the rescaled weights have no limit of their
    own, but the indicators -- squares of flux differences, with coefficients of order 1e4 in WENO7 -- overflow
    fp32): conserved values up to about 1e16 (WENO5) / 1e13 (WENO7).  The lumpy state times `scale` reaches about ten
    times that and must still give a finite L(u) that matches the fp64 oracle.  (Measured on the B200: WENO5 fails
    at scale 1e17, WENO7 at 1e14.)"""
    test_fp32_weno_weights_survive_any_data_scale(B, oracle, scheme, scale, 1e-6)


# ------------------------------------------------------------------ maximum sizes: index arithmetic beyond 2^31 elements
def test_large_noncubic_grid_beyond_2_31_elements(B, oracle):
    """1100 x 700 x 600 = 4.6e8 cells: one padded field has 4.7e8 elements, a state 2.4e9 (> 2^31) and 1.9e10 bytes
    (> 2^32), the workspace 57 GB.  The state is generated on the GPU (seeded torch generator; smooth hotspots with
    blended velocities like config 5), advanced by one WENO5 step, and checked on sampled cells against the oracle
    (19^3 crops, including cells in the last planes, rows and columns, whose offsets are the largest) and for
    conservation."""
    import torch
    nx, ny, nz = 1100, 700, 600
    free, _ = torch.cuda.mem_get_info()
    if free < 110e9:
        pytest.skip("needs about 110 GB of free device memory")
    dev, dt_ = "cuda", torch.float64
    g = torch.Generator(device=dev)
    g.manual_seed(1604)
    box = (nx / 32.0, ny / 32.0, nz / 32.0)
    dx = 1.0 / 32.0
    ax = [(torch.arange(n, device=dev, dtype=dt_) + 0.5) * dx for n in (nx, ny, nz)]
    X, Y, Z = ax[0].view(1, 1, nx), ax[1].view(1, ny, 1), ax[2].view(nz, 1, 1)
    e = torch.full((nz, ny, nx), 0.1, device=dev, dtype=dt_)
    mv = [torch.zeros_like(e) for _ in range(3)]
    nh = 24
    c = torch.rand(nh, 3, generator=g, device=dev, dtype=dt_) * torch.tensor(box, device=dev, dtype=dt_)
    sg = 0.6 + 1.0 * torch.rand(nh, generator=g, device=dev, dtype=dt_)
    A = torch.exp(0.5 * torch.randn(nh, generator=g, device=dev, dtype=dt_))
    vv = torch.randn(nh, 3, generator=g, device=dev, dtype=dt_)
    vv = vv / vv.norm(dim=1, keepdim=True) * (0.5 * torch.rand(nh, 1, generator=g, device=dev, dtype=dt_))
    for k in range(nh):
        def dist(a, cc, L):
            t = (a - cc).abs()
            return torch.minimum(t, L - t)
        gk = A[k] * (torch.exp(-dist(X, c[k, 0], box[0]) ** 2 / (2 * sg[k] ** 2)) *
                     torch.exp(-dist(Y, c[k, 1], box[1]) ** 2 / (2 * sg[k] ** 2)) *
                     torch.exp(-dist(Z, c[k, 2], box[2]) ** 2 / (2 * sg[k] ** 2)))
        e += gk
        for a in range(3):
            mv[a] += gk * vv[k, a]
        del gk
    cons = torch.empty((5, nz, ny, nx), device=dev, dtype=dt_)
    v2 = torch.zeros_like(e)
    for a in range(3):
        mv[a] /= e                      # blended velocity, |v| < 0.5
        v2 += mv[a] * mv[a]
    g2 = 1.0 / (1.0 - v2)
    del v2
    w = (4.0 / 3.0) * e * g2
    cons[0] = w - e / 3.0
    for a in range(3):
        cons[1 + a] = w * mv[a]
    cons[4] = 0.2 * e ** 0.75 * g2.sqrt()
    del w, g2, e, mv
    h = B.Hydro(nx, ny, nz, dx, W.WENO5)
    for axn in "xyz":
        h.set_option("bc_" + axn, W.BC_PERIODIC)
    h.bind()
    h.set_state(cons)
    dt = 0.2 * dx / h.max_signal_speed()
    tot0 = [float(cons[cc].sum()) for cc in range(5)]
    h.step(dt, 1)
    assert h.status() == 0
    out = h.get_state()
    tot1 = [float(out[cc].sum()) for cc in range(5)]
    for a, b in zip(tot0, tot1):
        assert abs(a - b) <= 1e-11 * abs(tot0[0]), (tot0, tot1)
    half = 9
    samples = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (nx - 2, 3, nz - 1), (30, ny - 1, 63), (31, 7, 64), (620, 127, 599),
               (nx // 2, ny // 2, nz // 2), (1099, 0, 128), (333, 699, 111)]
    scale = float(cons[0].abs().max())
    fmax = [float(cons[cc].abs().max()) for cc in range(5)]
    worst = 0.0
    for (i, j, k) in samples:
        ix = torch.arange(i - half, i + half + 1, device=dev) % nx
        iy = torch.arange(j - half, j + half + 1, device=dev) % ny
        iz = torch.arange(k - half, k + half + 1, device=dev) % nz
        crop = cons[:, iz][:, :, iy][:, :, :, ix].cpu().numpy()
        m = 2 * half + 1
        wc = W.Workload("crop", (m, m, m), dx, (0, 0, 0), W.WENO5, (W.BC_PERIODIC,) * 3, np.ascontiguousarray(crop))
        o = oracle.from_workload(wc)
        o.step(dt, 1)
        ref = o.get_state()[:, half, half, half]
        got = out[:, k, j, i].cpu().numpy()
        for cc in range(5):
            den = max(abs(ref[cc]), 1e-15 * scale) if cc == 0 else max(fmax[cc], 1e-15 * scale)
            worst = max(worst, abs(got[cc] - ref[cc]) / den)
    assert worst <= 3e-12, worst
    h.close()


def test_generic_kernel_must_be_chosen_before_the_workspace_is_bound(B):
    """The marching kernels keep no primitive arrays, so a workspace bound for them has none: asking for the generic
    kernel afterwards is refused (and leaves the context usable); asked for before the bind, it gets them."""
    w = small_workload(W.WENO5, (40, 33, 24))
    h = B.from_workload(w)
    n_fused = h.workspace_bytes()
    with pytest.raises(B.HydroError):
        h.set_option("kernel", B.KERNEL_GENERIC)
    h.step(1e-3, 1)
    assert h.status() == 0
    h.close()
    h2 = B.from_workload(w, kernel=B.KERNEL_GENERIC)
    assert h2.workspace_bytes() > n_fused
    h2.step(1e-3, 1)
    assert h2.status() == 0
    h2.close()
