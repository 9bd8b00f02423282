"""Slab decomposition along z: one exchange of g ghost planes per
Runge-Kutta stage with the two z-neighbours and one max-reduction of the signal speed per step.

Every step of the hot path runs in the library's kernels (hydro_get_zhalo / hydro_put_zhalo / hydro_local_max_speed /
hydro_step_stage_cfl); this module only routes device buffers between slabs -- the packed halo planes and the one
double of the signal-speed reduction -- and never brings a value to the host:

  * ``DistComm``   one slab per process, neighbours reached with torch.distributed point-to-point calls (NCCL on
                   GPUs; the same code runs over gloo on CPU tensors, which is how it is tested without GPUs);
  * ``LocalComm``  several slabs in ONE process on one GPU, advanced in lockstep: the emulation the profiling
                   guide asks for when there are fewer GPUs than ranks.  It is the parity test of the decomposition:
                   the result must be bit-identical to the undecomposed run.

A slab always runs with bc_z = BC_EXTERNAL; the periodic rule of the z axis is the ring closing, the outflow rule is
the library's (hydro_put_zhalo with no buffer: zero-gradient copies of the slab's own boundary plane).
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

    def exchange_async(self, pairs):
        """The same exchange issued on a side stream (CUDA tensors), so that the caller's stream is free to compute
        while the planes travel: returns (ghosts, event) with the event recorded on the side stream behind the
        receives; hydro_step_stage_overlap makes the compute stream wait for it only where the ghosts are needed.
        CPU tensors (gloo): a plain exchange, event None."""
        (send_lo, send_hi), = pairs
        if not send_lo.is_cuda:
            return self.exchange(pairs), None
        cur = torch.cuda.current_stream(send_lo.device)
        if getattr(self, "side", None) is None:
            self.side = torch.cuda.Stream(send_lo.device)
        self.side.wait_stream(cur)                       # the packing kernels have run
        with torch.cuda.stream(self.side):
            got = self.exchange(pairs)
            ready = torch.cuda.Event()
            ready.record(self.side)
        for t in (send_lo, send_hi):
            t.record_stream(self.side)                   # allocator: these buffers are in use on the side stream
        for t in got[0]:
            if t is not None:
                t.record_stream(cur)
        return got, ready

    def max(self, values):
        """values = [one 1-element float64 tensor] (this rank's slab): all-reduced in place with MAX over the ranks,
        on the tensor's device (NCCL on the GPU, gloo on the CPU); nothing comes to the host."""
        (t,) = values
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return t


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

    def exchange_async(self, pairs):
        return self.exchange(pairs), None

    def max(self, values):
        """Element-wise maximum of the slabs' 1-element tensors (what the all-reduce does between ranks)."""
        t = values[0]
        for v in values[1:]:
            t = torch.maximum(t, v)
        return t


class SlabGroup:
    """The slabs this process owns (one with DistComm, all of them with LocalComm) and the step loop."""

    def __init__(self, hydros, comm, dx):
        self.h, self.comm, self.dx = list(hydros), comm, dx
        for x in self.h:
            assert x.zhalo_elems() > 0

    def _fill_z_ghosts(self, buffer):
        pairs = [(x.get_zhalo(buffer, 0), x.get_zhalo(buffer, 1)) for x in self.h]
        got = self.comm.exchange(pairs)
        for x, (below, above) in zip(self.h, got):
            x.put_zhalo(buffer, 0, below)      # None at a physical end: the library's zero-gradient rule
            x.put_zhalo(buffer, 1, above)

    def step_cfl(self, cfl, nsteps=1, overlap=True):
        """Per step: the slabs' max signal speeds are max-reduced on the device, then three stages, each with a halo
        exchange; dt = cfl dx / max is taken inside the library.  No host sync.
        overlap: the exchange runs on a side stream while hydro_step_stage_overlap computes the planes that need no
        ghost; otherwise exchange -> hydro_put_zhalo -> hydro_step_stage_cfl one after the other.  Same results."""
        for _ in range(nsteps):
            a = self.comm.max([x.local_max_speed() for x in self.h])
            for s in range(3):
                if not overlap:
                    self._fill_z_ghosts(s)
                    for x in self.h:
                        x.step_stage_cfl(cfl, s, a)
                    continue
                pairs = [(x.get_zhalo(s, 0), x.get_zhalo(s, 1)) for x in self.h]
                got, ready = self.comm.exchange_async(pairs)
                for x, (below, above) in zip(self.h, got):
                    x.step_stage_overlap(cfl, s, a, below, above, ready)


def make_slab(binding, w, k0, k1, precision=0, device="cuda"):
    """Context for the z-range [k0, k1) of a workloads.Workload, bc_z = BC_EXTERNAL, state uploaded."""
    import numpy as np
    if binding.BC_HUBBLE in tuple(w.bc):
        # the closed-form ghosts need every Hubble axis and the slab's z position; the library refuses the
        # combination with bc_z = BC_EXTERNAL at step time, this says so before anything is uploaded
        raise ValueError("the slab decomposition does not support BC_HUBBLE (analytic ghost fill): %r" % (w.bc,))
    h = binding.Hydro(w.n[0], w.n[1], k1 - k0, w.dx, w.scheme, precision=precision, device=device)
    h.set_option("bc_x", w.bc[0])
    h.set_option("bc_y", w.bc[1])
    h.set_option("bc_z", binding.BC_EXTERNAL)
    for k, v in w.options.items():
        h.set_option(k, v)
    if getattr(w, "eos_table", None) is not None:
        h.set_eos_table(*w.eos_table)
    h.set_option("t", w.t0)
    h.bind()
    h.set_state(torch.from_numpy(np.ascontiguousarray(w.cons[:, k0:k1])).to(device=device, dtype=h.dtype).contiguous())
    return h
