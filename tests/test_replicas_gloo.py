"""The N > 1 path of bench.py is "replicas only": frames dealt to ranks, a barrier and a max over ranks
of the measured time.  Covered here with world_size 2 on the gloo backend (CPU)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1806_07938_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    replicas.barrier(world)
    mine = replicas.frames_of_rank(7, rank, world)
    t = replicas.max_over_ranks(10.0 + 5.0 * rank, world)          # the slowest rank defines the step time
    total = replicas.sum_over_ranks(float(len(mine)), world)       # units all ranks processed
    q.put((rank, mine, t, total))
    dist.destroy_process_group()


def test_two_replicas_share_frames_and_take_the_max_time():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0][1] == [0, 2, 4, 6] and got[1][1] == [1, 3, 5]
    assert all(g[2] == 15.0 and g[3] == 7.0 for g in got)


def test_frames_of_rank_partitions_exactly():
    for world in (1, 2, 3, 8):
        allf = sorted(f for r in range(world) for f in replicas.frames_of_rank(37, r, world))
        assert allf == list(range(37))
    with pytest.raises(ValueError):
        replicas.frames_of_rank(4, 2, 2)
