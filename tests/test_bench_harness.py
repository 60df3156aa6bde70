"""Host-side logic of bench.py's multi-rank path on CPU: world size 2 over gloo (no GPU needed).

The data path has no collective (frames are independent); what N > 1 adds is the
max-over-ranks timing, the per-rank frame offsets and the rule that only rank 0 runs the reference arm.
"""
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
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        slowest = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))
        # disjoint frame ranges, rank-major
        n = 7
        first = bench.first_frame_of_rank(rank, n)
        ranges = [None] * world
        dist.all_gather_object(ranges, (first, first + n))
        q.put((rank, slowest, ranges))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_frame_ranges_world2():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slowest, ranges in out:
        assert slowest == 15.0                       # both ranks report the slower rank's time
        assert ranges == [(0, 7), (7, 14)]           # weak scaling: each rank its own frames, no overlap


def test_single_rank_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, torch.device("cpu")) == 3.5
    assert bench.first_frame_of_rank(0, 100) == 0
