"""SURVEY 8(f)-N4 and N2 on the GPU: the CUDA-graph replay of hydro_step_cfl and the batched step of independent
contexts on their own streams must give, bit for bit, what the plain launches give -- and what the ORACLE gives when
it is advanced by the same rule (dt = cfl dx / max signal speed before every step, reading Q10), within 1e-10 in
fp64 (`-m gpu`)."""
import numpy as np
import pytest
import torch

from paper_1604_03360_b200 import workloads as W
from test_gpu_parity import SCHEMES, reldiff, small_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1604_03360_b200 import binding
    return binding


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("prec", [0, 1])
def test_graph_replay_is_bit_identical_to_plain_launches(B, oracle, scheme, prec):
    w = small_workload(scheme, (40, 33, 24))
    o = oracle.from_workload(w)
    oracle.run(o, w, nsteps=7)
    plain = B.from_workload(w, precision=prec)
    plain.step_cfl(0.2, 7)
    want, t_want, n_want = plain.get_state(), plain.time, plain.launch_count
    plain.close()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        h = B.from_workload(w, precision=prec)        # binds to the current (side) stream
        h.set_option("graph", 1)
        h.step_cfl(0.2, 1)                            # first step: plain launches (con2prim pass, max reduction)
        h.step_cfl(0.2, 2)                            # captures the graph of each buffer parity, replays
        h.step_cfl(0.2, 4)
        got = h.get_state()
        side.synchronize()
        assert h.status() == 0
        assert torch.equal(got, want)
        assert h.time == t_want
        assert reldiff(got.double().cpu().numpy(), o.get_state()) <= (1e-10 if prec == 0 else 1e-5)
        assert abs(h.time - o.time) <= (1e-12 if prec == 0 else 1e-5) * o.time
        assert h.launch_count == n_want               # the replayed launches are counted
        # an option change drops the graphs; the run goes on correctly
        h.set_option("weno_eps", 1e-6)
        h.step_cfl(0.2, 2)
        assert h.status() == 0
        h.close()


def test_graph_option_on_the_default_stream_falls_back(B):
    w = small_workload(W.WENO5, (40, 33, 24))
    ref = B.from_workload(w)
    ref.step_cfl(0.2, 4)
    h = B.from_workload(w)
    h.set_option("graph", 1)
    h.step_cfl(0.2, 4)
    assert torch.equal(h.get_state(), ref.get_state())
    ref.close()
    h.close()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_batched_events_equal_their_stand_alone_runs(B, oracle, scheme):
    """hydro_step_cfl_batch over three different events on three streams (one with the graph replay on): each event
    equals its stand-alone run bit for bit and the oracle's run of the same event within 1e-10."""
    ws = [small_workload(scheme, (40, 33, 24), seed=W.SEED + k) for k in range(3)]
    want, ref_o = [], []
    for w in ws:
        o = oracle.from_workload(w)
        oracle.run(o, w, nsteps=5)
        ref_o.append(o.get_state())
        h = B.from_workload(w)
        h.step_cfl(0.2, 5)
        want.append(h.get_state())
        h.close()
    streams = [torch.cuda.Stream() for _ in ws]
    hs = []
    for k, (w, st) in enumerate(zip(ws, streams)):
        with torch.cuda.stream(st):
            h = B.from_workload(w)
            if k == 1:
                h.set_option("graph", 1)
            hs.append(h)
    B.step_cfl_batch(hs, 0.2, 5)
    for h, st, ref, ro in zip(hs, streams, want, ref_o):
        with torch.cuda.stream(st):
            got = h.get_state()
        st.synchronize()
        assert h.status() == 0
        assert torch.equal(got, ref)
        assert reldiff(got.cpu().numpy(), ro) <= 1e-10
        h.close()
    assert not torch.equal(want[0], want[1])


def test_many_steps_from_one_graph_launch_in_pieces(B, oracle):
    """N4 as SURVEY 8(f) words it: the whole k-step loop of hydro_step_cfl from one graph launch (pieces of 64 steps).
    70 steps = one 64-step graph + one 6-step graph: bit-identical to 71 plain steps, same launch count, and the
    oracle's state within 1e-9."""
    w = small_workload(W.WENO5, (24, 20, 16))
    o = oracle.from_workload(w)
    oracle.run(o, w, nsteps=71)
    plain = B.from_workload(w)
    plain.step_cfl(0.2, 71)
    want, t_want, n_want = plain.get_state(), plain.time, plain.launch_count
    plain.close()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        h = B.from_workload(w)
        h.set_option("graph", 1)
        h.step_cfl(0.2, 1)
        h.step_cfl(0.2, 70)
        got = h.get_state()
        side.synchronize()
        assert torch.equal(got, want) and h.time == t_want and h.launch_count == n_want
        assert reldiff(got.cpu().numpy(), o.get_state()) <= 1e-9
        assert h.status() == 0
        h.close()
