"""Slab decomposition along z.  CPU: the partition and neighbour logic, and the
neighbour exchange / max-reduction over a 2-rank gloo group (the same code that runs over NCCL).  GPU (-m gpu):
several slabs advanced in lockstep in one process must reproduce the undecomposed run BIT FOR BIT."""
import math
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1604_03360_b200 import slab as S            # noqa: E402  (pure torch; loads no CUDA library)
from paper_1604_03360_b200 import workloads as W       # noqa: E402


def test_split_and_neighbours():
    assert S.split_planes(10, 3) == [(0, 4), (4, 7), (7, 10)]
    assert S.split_planes(512, 8)[-1] == (448, 512)
    assert S.neighbours(0, 4, S.BC_PERIODIC) == (3, 1) and S.neighbours(3, 4, S.BC_PERIODIC) == (2, 0)
    assert S.neighbours(0, 4, S.BC_OUTFLOW) == (None, 1) and S.neighbours(3, 4, S.BC_OUTFLOW) == (2, None)
    assert S.neighbours(0, 1, S.BC_PERIODIC) == (0, 0)


def test_local_comm_wiring():
    for bc in (S.BC_PERIODIC, S.BC_OUTFLOW):
        c = S.LocalComm(3, bc)
        pairs = [("lo%d" % r, "hi%d" % r) for r in range(3)]
        got = c.exchange(pairs)
        assert got[1] == ("hi0", "lo2")
        assert got[0] == (("hi2" if bc == S.BC_PERIODIC else None), "lo1")
        assert got[2] == ("hi1", ("lo0" if bc == S.BC_PERIODIC else None))
        assert float(c.max([torch.tensor([v], dtype=torch.float64) for v in (0.2, 0.7, 0.5)])) == 0.7


def _worker(rank, world, port, bc, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    comm = S.DistComm(dist, bc)
    lo = torch.full((6,), 10.0 * rank + 1.0, dtype=torch.float64)     # "my lowest planes"
    hi = torch.full((6,), 10.0 * rank + 2.0, dtype=torch.float64)     # "my highest planes"
    (below, above), = comm.exchange([(lo, hi)])
    m = float(comm.max([torch.tensor([0.3 + 0.1 * rank], dtype=torch.float64)]))
    out[rank] = (None if below is None else float(below[0]), None if above is None else float(above[0]), m)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("bc", [S.BC_PERIODIC, S.BC_OUTFLOW])
def test_dist_comm_over_gloo_two_ranks(bc):
    world, port = 2, 31500 + os.getpid() % 2000 + bc
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, bc, out), nprocs=world, join=True)
        res = dict(out)
    # rank 0's ghosts above are rank 1's lowest planes (11), rank 1's ghosts below are rank 0's highest (2)
    assert res[0][1] == 11.0 and res[1][0] == 2.0
    if bc == S.BC_PERIODIC:
        assert res[0][0] == 12.0 and res[1][1] == 1.0       # the ring closes
    else:
        assert res[0][0] is None and res[1][1] is None      # physical ends
    assert res[0][2] == res[1][2] == pytest.approx(0.4)


# ------------------------------------------------------------------ the whole control flow of SlabGroup.step_cfl off-GPU
class FakeHydro:
    """A CPU stand-in with the slab calls of binding.Hydro: one value per z-plane, g = 2 ghost planes, and a "stage"
    out = in + dt * (in[k-2] - 2 in[k] + in[k+2]) that needs BOTH ghost layers of the buffer it reads.  Stage s reads
    buffer s and writes buffer (s + 1) % 3, as the library does.  It only exists to drive SlabGroup."""
    G = 2

    def __init__(self, planes):
        self.nz = len(planes)
        self.shape = (5, self.nz, 1, 1)
        self.buf = [torch.zeros(self.nz + 2 * self.G, dtype=torch.float64) for _ in range(3)]
        self.buf[0][self.G:-self.G] = torch.as_tensor(planes, dtype=torch.float64)
        self.calls = []

    def zhalo_elems(self):
        return self.G

    def get_zhalo(self, buffer, side):
        v = self.buf[buffer][self.G:-self.G]
        return (v[:self.G] if side == 0 else v[-self.G:]).clone()

    def put_zhalo(self, buffer, side, packed):
        b = self.buf[buffer]
        if packed is None:      # zero-gradient
            packed = (b[self.G] if side == 0 else b[-self.G - 1]).repeat(self.G)
        if side == 0:
            b[:self.G] = packed
        else:
            b[-self.G:] = packed
        self.calls.append(("put", buffer, side))

    def local_max_speed(self):
        return self.buf[0][self.G:-self.G].abs().max().reshape(1).clone()

    def step_stage_cfl(self, cfl, stage, a):
        dt = cfl / float(a)
        u = self.buf[stage]
        G = self.G
        self.buf[(stage + 1) % 3][G:-G] = u[G:-G] + dt * (u[:-2 * G] - 2.0 * u[G:-G] + u[2 * G:])
        self.calls.append(("stage", stage))

    def step_stage_overlap(self, cfl, stage, a, lo, hi, ready):
        assert ready is None                      # CPU tensors: no stream to wait on
        self.put_zhalo(stage, 0, lo)
        self.put_zhalo(stage, 1, hi)
        self.step_stage_cfl(cfl, stage, a)

    def interior(self):
        return self.buf[0][self.G:-self.G].clone()


def _planes(nz):
    return [math.sin(0.7 * k) + 0.05 * k for k in range(nz)]


def _step_worker(rank, world, port, bc, nz, nsteps, overlap, out, bounds=None):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    k0, k1 = (bounds or S.split_planes(nz, world))[rank]
    h = FakeHydro(_planes(nz)[k0:k1])
    S.SlabGroup([h], S.DistComm(dist, bc), 1.0).step_cfl(0.1, nsteps, overlap=overlap)
    out[rank] = (h.interior().tolist(), h.calls[:9])
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("overlap", [False, True])
@pytest.mark.parametrize("bc", [S.BC_PERIODIC, S.BC_OUTFLOW])
def test_step_cfl_control_flow_over_gloo_two_ranks(bc, overlap):
    """SlabGroup.step_cfl end to end with two ranks over gloo: the max-reduction of the device scalar, one exchange
    per stage BEFORE that stage, the ring of two (periodic) or the zero-gradient ends (outflow).  The decomposed run
    must equal, bit for bit, the same fake advanced as one domain."""
    nz, nsteps, world = 11, 3, 2
    one = FakeHydro(_planes(nz))
    S.SlabGroup([one], S.LocalComm(1, bc), 1.0).step_cfl(0.1, nsteps, overlap=overlap)
    port = 33500 + os.getpid() % 2000 + bc + 2 * int(overlap)
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_step_worker, args=(world, port, bc, nz, nsteps, overlap, out), nprocs=world, join=True)
        res = dict(out)
    got = res[0][0] + res[1][0]
    assert got == one.interior().tolist()
    # per stage: both ghost sides of the stage's input buffer are written, then the stage runs
    assert res[0][1] == [("put", 0, 0), ("put", 0, 1), ("stage", 0), ("put", 1, 0), ("put", 1, 1), ("stage", 1),
                         ("put", 2, 0), ("put", 2, 1), ("stage", 2)]


@pytest.mark.parametrize("bc", [S.BC_PERIODIC, S.BC_OUTFLOW])
def test_very_unequal_slabs_over_gloo_two_ranks(bc):
    """The same with slabs of 8 and 3 planes (nothing in the exchange may assume equal slabs: a slab only ever sends
    and receives g planes per side) through the overlap call, zero-gradient ends or the ring of two."""
    nz, nsteps, world = 11, 4, 2
    one = FakeHydro(_planes(nz))
    S.SlabGroup([one], S.LocalComm(1, bc), 1.0).step_cfl(0.1, nsteps, overlap=True)
    port = 35600 + os.getpid() % 2000 + bc
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_step_worker, args=(world, port, bc, nz, nsteps, True, out, [(0, 8), (8, 11)]), nprocs=world, join=True)
        res = dict(out)
    assert len(res[0][0]) == 8 and len(res[1][0]) == 3
    assert res[0][0] + res[1][0] == one.interior().tolist()


# ------------------------------------------------------------------ GPU: bit-identity with the undecomposed run
@pytest.mark.gpu
@pytest.mark.parametrize("overlap", [False, True])
@pytest.mark.parametrize("scheme", [W.WENO5, W.WENO7, W.MUSTA_FORCE])
@pytest.mark.parametrize("bc_z,parts", [(W.BC_PERIODIC, 2), (W.BC_OUTFLOW, 3), (W.BC_PERIODIC, 1)])
def test_slabs_reproduce_the_single_domain_run_bit_for_bit(scheme, bc_z, parts, overlap):
    from paper_1604_03360_b200 import binding as B
    n = (40, 33, 70)
    big = W.lumpy(n=max(n), hotspots=12, with_velocity=True, scheme=scheme, box=max(n) / 16.0, sigma_unit=0.12)
    cons = np.ascontiguousarray(big.cons[:, :n[2], :n[1], :n[0]])
    w = W.Workload("slab", n, big.dx, (0.0, 0.0, 0.0), scheme, (W.BC_PERIODIC, W.BC_OUTFLOW, bc_z), cons, 0.0, cfl=0.2)
    ref = B.from_workload(w)
    ref.step_cfl(0.2, 3)
    want = ref.get_state().cpu()
    t_ref = ref.time
    ref.close()
    ranges = S.split_planes(n[2], parts)
    hs = [S.make_slab(B, w, k0, k1) for k0, k1 in ranges]
    group = S.SlabGroup(hs, S.LocalComm(parts, bc_z), w.dx)
    group.step_cfl(0.2, 3, overlap=overlap)
    got = torch.cat([h.get_state().cpu() for h in hs], dim=1)
    assert all(h.status() == 0 for h in hs)
    assert abs(hs[0].time - t_ref) == 0.0
    assert torch.equal(got, want)
    for h in hs:
        h.close()


@pytest.mark.gpu
@pytest.mark.parametrize("scheme", [W.WENO5, W.WENO7, W.MUSTA_FORCE])
@pytest.mark.parametrize("n", [(1, 24, 30), (40, 33, 24)])
def test_generic_kernel_slabs_with_overlap_call(scheme, n):
    """The slab calls on the generic kernel (a grid with an inactive axis, or "kernel" = generic): the overlap call
    has nothing to split there, but must still give the undecomposed result bit for bit."""
    from paper_1604_03360_b200 import binding as B
    cons = W.random_state((n[2], n[1], n[0]), seed=9, vmax=0.4)
    w = W.Workload("g", n, 0.05, (0.0, 0.0, 0.0), scheme, (W.BC_PERIODIC, W.BC_OUTFLOW, W.BC_PERIODIC), cons, 0.0, cfl=0.2,
                   options={"kernel": 1})
    ref = B.from_workload(w, kernel=B.KERNEL_GENERIC)
    ref.step_cfl(0.2, 3)
    want = ref.get_state().cpu()
    ref.close()
    for overlap in (True, False):
        hs = [S.make_slab(B, w, k0, k1) for k0, k1 in S.split_planes(n[2], 2)]
        S.SlabGroup(hs, S.LocalComm(2, W.BC_PERIODIC), w.dx).step_cfl(0.2, 3, overlap=overlap)
        got = torch.cat([h.get_state().cpu() for h in hs], dim=1)
        assert torch.equal(got, want)
        for h in hs:
            h.close()


@pytest.mark.gpu
@pytest.mark.parametrize("scheme,g", [(W.WENO5, 3), (W.MUSTA_FORCE, 2)])
def test_put_zhalo_without_a_buffer_is_the_outflow_rule(scheme, g):
    """hydro_put_zhalo(NULL) on a slab with external z ghosts must give exactly what bc_z = outflow gives: the same
    L(u)-driven step, bit for bit (reading Q9 applied by the library, not by the Python side)."""
    from paper_1604_03360_b200 import binding as B
    n = (24, 17, 15)
    big = W.lumpy(n=max(n), hotspots=12, with_velocity=True, scheme=scheme, box=max(n) / 16.0, sigma_unit=0.12)
    cons = np.ascontiguousarray(big.cons[:, :n[2], :n[1], :n[0]])
    w = W.Workload("slab", n, big.dx, (0.0, 0.0, 0.0), scheme, (W.BC_PERIODIC, W.BC_OUTFLOW, W.BC_OUTFLOW), cons, 0.0)
    ref = B.from_workload(w)
    ref.step(1e-3, 2)
    want = ref.get_state().cpu()
    ref.close()
    h = S.make_slab(B, w, 0, n[2])
    for _ in range(2):
        for s in range(3):
            h.put_zhalo(s, 0, None)
            h.put_zhalo(s, 1, None)
            h.step_stage(1e-3, s)
    assert torch.equal(h.get_state().cpu(), want)
    h.close()


@pytest.mark.gpu
@pytest.mark.parametrize("scheme", [W.WENO5, W.MUSTA_FORCE])
def test_dist_comm_side_stream_path_on_one_gpu(scheme):
    """DistComm over a one-rank NCCL group (a periodic ring of one): the exchange is issued on the side stream, the
    stage waits for its event only before the boundary planes; the result must equal the undecomposed run bit for
    bit, and the serial (no overlap) path too."""
    from paper_1604_03360_b200 import binding as B
    dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % (36500 + os.getpid() % 2000 + scheme), rank=0,
                            world_size=1)
    try:
        _ring_of_one(B, scheme)
    finally:
        dist.destroy_process_group()


def _ring_of_one(B, scheme):
    n = (40, 33, 70)
    big = W.lumpy(n=max(n), hotspots=12, with_velocity=True, scheme=scheme, box=max(n) / 16.0, sigma_unit=0.12)
    cons = np.ascontiguousarray(big.cons[:, :n[2], :n[1], :n[0]])
    w = W.Workload("ring1", n, big.dx, (0.0, 0.0, 0.0), scheme, (W.BC_PERIODIC,) * 3, cons, 0.0, cfl=0.2)
    ref = B.from_workload(w)
    ref.step_cfl(0.2, 4)
    want = ref.get_state()
    ref.close()
    for overlap in (True, False):
        h = S.make_slab(B, w, 0, n[2])
        S.SlabGroup([h], S.DistComm(dist, W.BC_PERIODIC), w.dx).step_cfl(0.2, 4, overlap=overlap)
        assert torch.equal(h.get_state(), want)
        assert h.status() == 0
        h.close()


def test_make_slab_refuses_the_analytic_ghost_fill():
    """BC_HUBBLE needs all its axes and the slab's z position; a slab would get silently wrong ghosts."""
    class FakeBinding:
        BC_HUBBLE, BC_EXTERNAL = 2, 3

        def Hydro(self, *a, **k):
            raise AssertionError("the check comes before the context is made")
    w = W.hubble(n=8)
    assert W.BC_HUBBLE in w.bc
    with pytest.raises(ValueError, match="BC_HUBBLE"):
        S.make_slab(FakeBinding(), w, 0, 4)


@pytest.mark.gpu
@pytest.mark.parametrize("scheme", [W.WENO5, W.MUSTA_FORCE])
def test_library_refuses_hubble_ghosts_on_a_slab(scheme):
    """The same rule inside the library: every stepping call of a context with bc_z = EXTERNAL and a Hubble axis
    returns EINVAL, and the plain combination still runs."""
    import torch
    from paper_1604_03360_b200 import binding as B
    h = B.Hydro(16, 16, 16, 0.1, scheme, bc_x=B.BC_HUBBLE, bc_y=B.BC_OUTFLOW, bc_z=B.BC_EXTERNAL).bind()
    cons = torch.from_numpy(W.random_state((16, 16, 16), seed=3)).cuda().contiguous()
    h.set_state(cons)
    a = torch.ones(1, dtype=torch.float64, device="cuda")
    for call in (lambda: h.step_stage(0.01, 0), lambda: h.step_stage_cfl(0.2, 0, a),
                 lambda: h.step_stage_overlap(0.2, 0, a, None, None), lambda: h.step(0.01), lambda: h.eval_L(cons)):
        with pytest.raises(B.HydroError) as e:
            call()
        assert e.value.code == B.EINVAL and "HYDRO_BC_HUBBLE" in str(e.value)
    h.set_option("bc_x", B.BC_PERIODIC)
    h.put_zhalo(0, 0, None)
    h.put_zhalo(0, 1, None)
    h.step_stage(0.01, 0)          # accepted (the rough random state may raise the clamp flag: not the point here)
    torch.cuda.synchronize()
    h.close()
