"""The N > 1 path is replicas only: world_size-2 gloo test of its host logic — the round-robin dealing
of the 12 propagator columns and the max-over-ranks reduction of a per-rank time."""
import os
import socket

import pytest

from paper_2201_09004_b200 import columns

torch = pytest.importorskip("torch")


def test_columns_partition_exactly():
    for world in (1, 2, 3, 4, 6, 8, 12):
        dealt = [c for r in range(world) for c in columns.columns_for_rank(r, world)]
        if world <= 12 and 12 % world == 0:
            assert sorted(dealt) == list(range(12))
        assert set(dealt) == set(range(12)) or world > 12
    assert columns.columns_for_rank(13, 16) == [1]
    assert columns.spin_colour(7) == (2, 1)
    with pytest.raises(ValueError):
        columns.columns_for_rank(2, 2)


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cols = columns.columns_for_rank(rank, world)
        ms = columns.max_over_ranks(10.0 + 5.0 * rank, dist)
        gathered = [None] * world
        dist.all_gather_object(gathered, cols)
        q.put((rank, cols, ms, gathered))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == [0, 2, 4, 6, 8, 10] and res[1][1] == [1, 3, 5, 7, 9, 11]
    assert res[0][2] == res[1][2] == 15.0  # max over ranks
    assert sorted(res[0][3][0] + res[0][3][1]) == list(range(12))
