"""N > 1 path of bench.py on the CPU: two `gloo` ranks (the path is "replicas only", DESIGN.md
section 8: independent solves, one per GPU, no data-path collective; the only exchange is the
max-over-ranks time and the summed counts)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    sys.path.insert(0, ROOT)
    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r: r-dependent figures, so that max and sum are distinguishable from either rank's own
    res = bench.aggregate_over_ranks(world, torch.device("cpu"), ms=100.0 + 7 * rank, e_ms=200.0 - 5 * rank,
                                     iters=1000 + rank, e_iters=2000 + 3 * rank, launches=50 * (rank + 1))
    dist.barrier()
    out[rank] = res
    dist.destroy_process_group()


def test_two_rank_aggregation_max_time_summed_counts():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0 == r1  # every rank holds the job-wide figures; rank 0 prints them
    ms, e_ms, iters, e_iters, launches = r0
    assert ms == 107.0 and e_ms == 200.0          # max over ranks
    assert iters == 2001 and e_iters == 4003      # summed: whole-job iterations
    assert launches == 150


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.aggregate_over_ranks(1, torch.device("cpu"), 1.5, 2.5, 3, 4, 5) == (1.5, 2.5, 3, 4, 5)
