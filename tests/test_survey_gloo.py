"""Not gpu: the N > 1 host logic (shot partition, image stacking, max-over-ranks timing) with the gloo
backend, world_size 2, on CPU."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2201_06914_b200.survey import max_over_ranks, partition_shots, stack_across_ranks


def test_partition_covers_every_shot_once():
    for nshots in (0, 1, 5, 44, 71):
        for world in (1, 2, 3, 8):
            got = [i for r in range(world) for i in partition_shots(nshots, world, r)]
            assert got == list(range(nshots))
            sizes = [len(partition_shots(nshots, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        partition_shots(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, nshots, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = partition_shots(nshots, world, rank)
        img = torch.zeros(6, 5)
        for s in mine:                      # stand-in for one migrated shot: a rank-independent contribution
            img += torch.full((6, 5), float(s + 1))
        stack_across_ranks(img)
        t = max_over_ranks(10.0 + rank)
        q.put((rank, img.clone(), t, list(mine)))
    finally:
        dist.destroy_process_group()


def test_stack_and_timing_world2():
    world, nshots = 2, 7
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, nshots, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    expect = float(sum(range(1, nshots + 1)))
    seen = []
    for rank, img, t, mine in res:
        assert torch.all(img == expect)
        assert t == 11.0
        seen += mine
    assert sorted(seen) == list(range(nshots))
