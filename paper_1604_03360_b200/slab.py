"""Slab decomposition along z: one exchange of g ghost planes per
Runge-Kutta stage with the two z-neighbours and one max-reduction of the signal speed per step.

Every step of the hot path runs in the library's kernels (hydro_get_zhalo / hydro_put_zhalo / hydro_step_stage);
this module only moves the packed halo buffers between slabs:

  * ``DistComm``   one slab per process, neighbours reached with torch.distributed point-to-point calls (NCCL on
                   GPUs; the same code runs over gloo on CPU tensors, which is how it is tested without GPUs);
  * ``LocalComm``  several slabs in ONE process on one GPU, advanced in lockstep: the emulation the profiling
                   guide asks for when there are fewer GPUs than ranks.  It is the parity test of the decomposition:
                   the result must be bit-identical to the undecomposed run.

The physical boundary rule of the z axis (periodic or outflow) is applied here, on the packed buffers: a slab
always runs with bc_z = BC_EXTERNAL.
"""
from __future__ import annotations

import torch

BC_OUTFLOW, BC_PERIODIC = 0, 1


def split_planes(nz, parts):
    """Contiguous z-ranges [(k0, k1), ...] of `parts` slabs, sizes differing by at most one plane."""
    base, extra = divmod(nz, parts)
    out, k = [], 0
    for r in range(parts):
        n = base + (1 if r < extra else 0)
        out.append((k, k + n))
        k += n
    return out


def neighbours(rank, world, bc_z):
    """(lower, upper) neighbour ranks of a slab; None at a physical (outflow) end."""
    lo = rank - 1 if rank > 0 else (world - 1 if bc_z == BC_PERIODIC else None)
    hi = rank + 1 if rank < world - 1 else (0 if bc_z == BC_PERIODIC else None)
    return lo, hi


def outflow_ghost(own_planes, g, side):
    """Zero-gradient ghost planes from a slab's own packed boundary planes [5][g][ny][nx] (reading Q9): every
    ghost layer repeats the nearest interior plane (the lowest one for side 0, the highest for side 1)."""
    v = own_planes.view(5, g, -1)
    src = v[:, 0:1] if side == 0 else v[:, g - 1:g]
    return src.expand(5, g, v.shape[2]).contiguous().view(-1)


class DistComm:
    """Neighbour exchange and max-reduction over a torch.distributed process group (one slab per rank)."""

    def __init__(self, dist, bc_z):
        self.dist, self.bc_z = dist, bc_z
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.lo, self.hi = neighbours(self.rank, self.world, bc_z)

    def exchange(self, pairs):
        """pairs = [(my lowest planes, my highest planes)] (one local slab) -> [(ghosts below, ghosts above)];
        an entry is None at a physical end."""
        (send_lo, send_hi), = pairs
        recv_lo = torch.empty_like(send_lo) if self.lo is not None else None
        recv_hi = torch.empty_like(send_hi) if self.hi is not None else None
        if self.world == 1:
            # a periodic ring of one: the slab is its own neighbour
            return [(send_hi.clone() if self.lo is not None else None, send_lo.clone() if self.hi is not None else None)]
        # order matters when both neighbours are the same rank (periodic ring of two): my upward message is my
        # peer's first receive (its ghosts below), my downward message its second (its ghosts above)
        P2P = self.dist.P2POp
        ops = []
        if self.hi is not None:
            ops.append(P2P(self.dist.isend, send_hi, self.hi))
        if self.lo is not None:
            ops.append(P2P(self.dist.irecv, recv_lo, self.lo))
            ops.append(P2P(self.dist.isend, send_lo, self.lo))
        if self.hi is not None:
            ops.append(P2P(self.dist.irecv, recv_hi, self.hi))
        for req in self.dist.batch_isend_irecv(ops):
            req.wait()
        return [(recv_lo, recv_hi)]

    def max(self, values):
        t = torch.tensor([max(values)], dtype=torch.float64)
        if self.world > 1:
            dev = "cuda" if self.dist.get_backend() == "nccl" else "cpu"
            t = t.to(dev)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())


class LocalComm:
    """All slabs live in this process (in z order): neighbours are list neighbours."""

    def __init__(self, nslabs, bc_z):
        self.n, self.bc_z = nslabs, bc_z

    def exchange(self, pairs):
        out = []
        for r in range(self.n):
            lo, hi = neighbours(r, self.n, self.bc_z)
            out.append((pairs[lo][1] if lo is not None else None, pairs[hi][0] if hi is not None else None))
        return out

    def max(self, values):
        return max(values)


class SlabGroup:
    """The slabs this process owns (one with DistComm, all of them with LocalComm) and the step loop."""

    def __init__(self, hydros, comm, dx):
        self.h, self.comm, self.dx = list(hydros), comm, dx
        for x in self.h:
            assert x.zhalo_elems() > 0

    def _fill_z_ghosts(self, buffer):
        g_elems = [x.zhalo_elems() for x in self.h]
        pairs = [(x.get_zhalo(buffer, 0), x.get_zhalo(buffer, 1)) for x in self.h]
        got = self.comm.exchange(pairs)
        for x, (own_lo, own_hi), (below, above), ne in zip(self.h, pairs, got, g_elems):
            g = ne // (5 * x.shape[2] * x.shape[3])
            x.put_zhalo(buffer, 0, below if below is not None else outflow_ghost(own_lo, g, 0))
            x.put_zhalo(buffer, 1, above if above is not None else outflow_ghost(own_hi, g, 1))

    def step_cfl(self, cfl, nsteps=1):
        """dt = cfl dx / (max signal speed over ALL slabs), then three stages, each after a halo exchange."""
        dts = []
        for _ in range(nsteps):
            a = self.comm.max([x.max_signal_speed() for x in self.h])
            dt = cfl * self.dx / a
            for s in range(3):
                self._fill_z_ghosts(s)
                for x in self.h:
                    x.step_stage(dt, s)
            dts.append(dt)
        return dts


def make_slab(binding, w, k0, k1, precision=0, device="cuda"):
    """Context for the z-range [k0, k1) of a workloads.Workload, bc_z = BC_EXTERNAL, state uploaded."""
    import numpy as np
    h = binding.Hydro(w.n[0], w.n[1], k1 - k0, w.dx, w.scheme, precision=precision, device=device)
    h.set_option("bc_x", w.bc[0])
    h.set_option("bc_y", w.bc[1])
    h.set_option("bc_z", binding.BC_EXTERNAL)
    for k, v in w.options.items():
        h.set_option(k, v)
    h.set_option("t", w.t0)
    h.bind()
    h.set_state(torch.from_numpy(np.ascontiguousarray(w.cons[:, k0:k1])).to(device=device, dtype=h.dtype).contiguous())
    return h
