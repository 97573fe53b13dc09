"""The N > 1 path of bench.py (replicas + barrier + max-over-ranks timing), exercised with 2 gloo processes on CPU."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2409_10327_b200 import dist as hd
    assert hd.world() == (rank, world)
    hd.barrier()
    ms = hd.max_over_ranks(10.0 + 5.0 * rank)            # rank 1 is slower: 15 ms
    rate = hd.whole_job_rate(450_560_000, ms)
    hd.barrier()
    q.put((rank, ms, rate))
    dist.destroy_process_group()


def test_two_rank_timing_protocol():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, rate in out:
        assert ms == 15.0                                   # max over ranks, seen by every rank
        assert rate == 2 * 450_560_000 / 15e-3              # whole-job aggregate of two replicas


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    from paper_2409_10327_b200 import dist as hd
    assert hd.world() == (0, 1)
    assert hd.max_over_ranks(3.5) == 3.5
    assert hd.whole_job_rate(100, 10.0) == 100 / 10e-3
