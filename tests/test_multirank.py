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
    # one image dealt out in tiles: every rank holds values of its own rays only, in shard
    # order; after the gather every rank holds the whole image in ray order
    n, tile = 1003, 64                                    # 16 tiles, the last one ragged
    mine = multi.shard_global_index(n, tile, rank, world)
    local = torch.stack([mine.double() * 3.0 + 1.0, -mine.double()])       # (2, n_local): "results" of my rays
    full = multi.gather_image(local, n, tile)
    local_i = (mine % 5).to(torch.int32)                                     # a status-like integer array
    full_i = multi.gather_image(local_i, n, tile)
    if rank == 0:
        torch.save({"times": times, "work": work, "full": full, "full_i": full_i, "n_local": mine.numel()}, out)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_reduction_and_sharding(tmp_path):
    out = str(tmp_path / "r.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    res = torch.load(out)
    assert res["times"] == [2.0, 0.5]          # max over ranks
    assert res["work"] == [1001.0, 30.0]       # sum over ranks: the shards tile the units exactly
    g = torch.arange(1003, dtype=torch.float64)
    assert torch.equal(res["full"], torch.stack([g * 3.0 + 1.0, -g]))
    assert torch.equal(res["full_i"], (torch.arange(1003) % 5).to(torch.int32))
    assert res["n_local"] == 8 * 64            # rank 0 owns tiles 0, 2, ..., 14 (the ragged tile 15 is rank 1's)


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


def test_tile_dealing_is_a_permutation_and_matches_the_library_count():
    sys.path.insert(0, ROOT)
    import ctypes as C
    from paper_1706_07062_b200 import build, multi
    lib = C.CDLL(build.build())
    lib.gray2_shard_count.argtypes = [C.c_uint64, C.c_uint64, C.c_int32, C.c_int32]
    lib.gray2_shard_count.restype = C.c_uint64
    for n, tile, world in ((10, 3, 2), (4096, 4096, 3), (1000, 7, 3), (5, 10, 4), (1 << 20, 4096, 8), (77, 1, 5)):
        parts = [multi.shard_global_index(n, tile, r, world) for r in range(world)]
        assert sorted(torch.cat(parts).tolist()) == list(range(n))
        for r, p in enumerate(parts):
            assert lib.gray2_shard_count(n, tile, r, world) == p.numel()
            # the formula of gray2_init_null_shard
            j = torch.arange(p.numel())
            assert torch.equal(p, ((j // tile) * world + r) * tile + j % tile)
    assert lib.gray2_shard_count(10, 0, 0, 1) == 0 and lib.gray2_shard_count(10, 3, 2, 2) == 0    # bad arguments


def _bench_rank(payload):
    """What bench.py's ranks do around the measurement, on CPU: read the torchrun-style environment that
    launch_ranks sets, join the group, reduce (time = max, work = sum)."""
    sys.path.insert(0, ROOT)
    from paper_1706_07062_b200 import multi
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    assert int(os.environ["LOCAL_RANK"]) == rank and os.environ["MASTER_ADDR"] == "127.0.0.1"
    dist.init_process_group("gloo")
    times, work = multi.reduce_job([0.25 * (rank + 1)], [100 + rank])
    if rank == 0:
        torch.save({"times": times, "work": work, "world": world}, payload)
    dist.barrier()
    dist.destroy_process_group()
    return 0


def _failing_rank(payload):
    return 3 if int(os.environ["RANK"]) == 1 else 0


def test_bench_launch_ranks_starts_n_processes_with_the_torchrun_environment(tmp_path):
    import bench                                            # bench.py at the repo root (conftest puts it on sys.path)
    out = str(tmp_path / "b.pt")
    assert bench.launch_ranks(2, _bench_rank, out) == 0
    res = torch.load(out)
    assert res == {"times": [0.5], "work": [201.0], "world": 2}
    import pytest
    with pytest.raises(Exception):
        bench.launch_ranks(2, _failing_rank, None)          # a failing rank fails the launch
