"""world_size-2 test (gloo, CPU) of the multi-rank protocol bench.py uses: replicas only, barrier on
both sides, MAX over ranks of the measured time, whole-job throughput = all ranks' units / that time."""
import os
import socket

import torch
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1301_5892_b200 import multi
    r, w = multi.init("gloo")
    assert (r, w) == (rank, world)
    multi.barrier()
    ms_local = 10.0 * (rank + 1)                 # rank 1 is the slow one
    ms = multi.max_over_ranks(ms_local)
    thr = multi.aggregate_throughput(1000, w, ms)
    out[rank] = (ms, thr)
    multi.finalize()


def test_two_rank_timing_protocol():
    world = 2
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms, thr = res[0]
    assert ms == 20.0
    assert abs(thr - 2 * 1000 / 0.020) < 1e-6


def test_single_rank_is_a_no_op():
    from paper_1301_5892_b200 import multi
    assert multi.max_over_ranks(3.5) == 3.5
    assert multi.aggregate_throughput(100, 1, 50.0) == 2000.0
