"""The N > 1 path on CPU: two gloo ranks exercise the sharding and the max-time / sum-work reductions
that bench.py uses (the data path itself has no collective: geodesics are independent)."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    from paper_1706_07062_b200 import multi
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = multi.shard_range(1001, rank, world)
    times, work = multi.reduce_job([1.0 + rank, 0.5], [hi - lo, 10 * (rank + 1)])
    if rank == 0:
        torch.save({"times": times, "work": work}, out)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_reduction_and_sharding(tmp_path):
    out = str(tmp_path / "r.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    res = torch.load(out)
    assert res["times"] == [2.0, 0.5]          # max over ranks
    assert res["work"] == [1001.0, 30.0]       # sum over ranks: the shards tile the units exactly


def test_shard_range_tiles_exactly():
    sys.path.insert(0, ROOT)
    from paper_1706_07062_b200 import multi
    for n in (0, 1, 7, 1024, 1048576 + 3):
        for world in (1, 2, 3, 8):
            pieces = [multi.shard_range(n, r, world) for r in range(world)]
            assert pieces[0][0] == 0 and pieces[-1][1] == n
            assert all(pieces[i][1] == pieces[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in pieces]
            assert max(sizes) - min(sizes) <= 1
    assert multi.reduce_job([3.0], [5]) == ([3.0], [5.0])    # single process: identity
