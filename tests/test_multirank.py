"""The N > 1 path of bench.py on CPU: world_size 2 over gloo.  Every rank advances its own independent event
(no data-path collective); what crosses ranks is the max-over-ranks of the timing and
the aggregate throughput.  Also checks that ranks draw different events from the seeded generator."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, dist, "cpu")
    w = bench.make_workload(64, "weno5", rank)
    # cross-check that the ranks hold different events: all-gather one scalar fingerprint
    fp = torch.tensor([float(w.cons[0].sum())], dtype=torch.float64)
    got = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(got, fp)
    out[rank] = (ms, bench.aggregate_value(64 ** 3, 4, world, ms), [float(g) for g in got])
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_max_time_and_aggregate_value():
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in (0, 1):
        ms, value, fps = res[rank]
        assert ms == 15.0                                # the max over ranks, on every rank
        assert value == 64 ** 3 * 4 * 2 / 15.0e-3        # both events count, divided by the slowest rank's time
        assert fps[0] != fps[1]                          # different seeded events per rank
    assert res[0][2] == res[1][2]


def test_single_process_is_the_identity():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.aggregate_value(1000, 2, 1, 4.0) == 1000 * 2 / 4.0e-3
