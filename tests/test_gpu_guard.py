"""Memory-safety and race checks of the CUDA path without compute-sanitizer (which is closed on this GPU pool):
  * every buffer the library is given (workspace, state in, state out, L out, packed z halos) sits between two guard
    regions filled with a byte pattern; after set_state / eval_L / steps / get_state on ragged grids with short march
    chunks the guards must be untouched (an out-of-bounds store would hit them: the marching kernels address with
    halo offsets on every side of the padded arrays);
  * the same run done twice must give bit-identical results (a shared-memory or global race between the warps of the
    barrier-free marching kernels would show up as run-to-run differences), and the parity tests against the oracle
    (tests/test_gpu_parity.py, tests/test_gpu_seams.py) bound every value."""
import ctypes

import numpy as np
import pytest
import torch

from paper_1604_03360_b200 import workloads as W
from test_gpu_parity import SCHEMES, small_workload

pytestmark = pytest.mark.gpu
GUARD = 1 << 20
PATTERN = 0xA5


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1604_03360_b200 import binding
    return binding


class Guarded:
    """nbytes of device memory (256-byte aligned) between two guard regions."""

    def __init__(self, nbytes):
        self.raw = torch.full((nbytes + 2 * GUARD + 256,), PATTERN, dtype=torch.uint8, device="cuda")
        base = self.raw.data_ptr()
        self.off = (base + GUARD + 255) // 256 * 256 - base
        self.nbytes = nbytes
        self.ptr = base + self.off

    def view(self, dtype, shape):
        return self.raw[self.off:self.off + self.nbytes].view(dtype).view(shape)

    def intact(self):
        lo = self.raw[:self.off]
        hi = self.raw[self.off + self.nbytes:]
        return bool((lo == PATTERN).all().item()) and bool((hi == PATTERN).all().item())


def _run(B, w, prec, chunks):
    dtype = torch.float32 if prec else torch.float64
    esz = 4 if prec else 8
    h = B.Hydro(w.n[0], w.n[1], w.n[2], w.dx, w.scheme, precision=prec)
    for ax, b in zip("xyz", w.bc):
        h.set_option("bc_" + ax, b)
    h.set_option("tile_zc", chunks[0])
    h.set_option("sweep_zc", chunks[1])
    ws = Guarded(h.workspace_bytes())
    h._check(B.lib.hydro_set_stream(h._h, torch.cuda.current_stream().cuda_stream))
    h._check(B.lib.hydro_bind_workspace(h._h, ws.ptr, ws.nbytes))
    nstate = 5 * w.n[0] * w.n[1] * w.n[2] * esz
    gin, gout, gL = Guarded(nstate), Guarded(nstate), Guarded(nstate)
    shape = (5, w.n[2], w.n[1], w.n[0])
    gin.view(dtype, shape).copy_(torch.from_numpy(w.cons).to(dtype))
    h._check(B.lib.hydro_set_state(h._h, gin.ptr))
    guards = [ws, gin, gout, gL]
    if w.bc[2] == B.BC_EXTERNAL:
        # the slab protocol: ghost planes of every stage input come from the caller -- here the slab's own opposite
        # boundary planes through a guarded packed buffer (a periodic ring of one) and the zero-gradient rule
        gh = Guarded(h.zhalo_elems() * esz)
        guards.append(gh)
        for step in range(2):
            for s in range(3):
                h._check(B.lib.hydro_get_zhalo(h._h, s, 1, gh.ptr))
                h._check(B.lib.hydro_put_zhalo(h._h, s, 0, gh.ptr))
                h._check(B.lib.hydro_put_zhalo(h._h, s, 1, None))
                h.step_stage(1e-3, s)
        L = None
    else:
        h._check(B.lib.hydro_eval_L(h._h, gin.ptr, 0.0, gL.ptr))
        h.step_cfl(0.2, 2)
        h.step(1e-3, 1)
    h._check(B.lib.hydro_get_state(h._h, gout.ptr))
    torch.cuda.synchronize()
    out = gout.view(dtype, shape).clone()
    Lout = gL.view(dtype, shape).clone()
    ok = all(g.intact() for g in guards)
    h.close()
    return out, Lout, ok


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("n,chunks", [((70, 45, 40), (5, 7)), ((33, 5, 9), (64, 128)), ((31, 4, 3), (1, 1)),
                                      ((150, 37, 29), (16, 16))])
def test_no_store_outside_the_buffers_and_runs_repeat_bit_for_bit(B, scheme, prec, n, chunks):
    g = {W.WENO5: 3, W.WENO7: 4, W.MUSTA_FORCE: 2}[scheme]
    n = tuple(max(v, g) for v in n)
    for bc in ((W.BC_PERIODIC,) * 3, (W.BC_OUTFLOW, W.BC_PERIODIC, B.BC_EXTERNAL)):
        w = small_workload(scheme, n)
        w.bc = bc
        a, La, ok_a = _run(B, w, prec, chunks)
        b, Lb, ok_b = _run(B, w, prec, chunks)
        assert ok_a and ok_b, "a kernel wrote outside a buffer it was given"
        assert torch.isfinite(a).all() and torch.isfinite(La).all()
        assert torch.equal(a, b) and torch.equal(La, Lb), "two identical runs differ: a race"


def test_inactive_axes_keep_inside_their_buffers(B):
    """The generic kernel (400 x 1 x 1 shock-tube shape and a 2-D sheet) with its primitive array."""
    for n in ((97, 1, 1), (1, 41, 23)):
        cons = W.random_state((n[2], n[1], n[0]), seed=5, vmax=0.5)
        w = W.Workload("thin", n, 0.05, (0, 0, 0), W.WENO5, (W.BC_OUTFLOW,) * 3, cons)
        a, La, ok = _run(B, w, 0, (64, 128))
        b, Lb, ok2 = _run(B, w, 0, (64, 128))
        assert ok and ok2 and torch.equal(a, b) and torch.equal(La, Lb)
