"""The N > 1 plumbing on CPU: world_size 2 over gloo (rank ownership of batches, MAX-over-ranks timing)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1408_0698_b200.distributed import job_throughput, max_over_ranks, rank_batches, rank_frames


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = 10.0 + 5.0 * rank                                # rank 1 is slower
        worst = max_over_ranks(ms)
        frames = list(rank_frames(1000, 100, rank, world))
        gathered = [None] * world
        dist.all_gather_object(gathered, frames)
        q.put((rank, worst, frames, gathered))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_max_time_and_disjoint_batches():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, worst, frames, gathered in res:
        assert worst == 15.0                                  # MAX over ranks, on every rank
        assert frames == list(range(rank * 100, rank * 100 + 100))
        assert not set(gathered[0]) & set(gathered[1])        # ranks own different batches
    assert job_throughput(1000, 10, 15.0, 2) == pytest.approx(2 * 1000 * 10 / 0.015)


def test_rank_batches_cover_the_stream_once():
    for world in (1, 2, 4, 8):
        seen = sorted(b for r in range(world) for b in rank_batches(10, r, world))
        assert seen == list(range(10))
    with pytest.raises(ValueError):
        rank_batches(10, 3, 2)
    assert max_over_ranks(3.5) == 3.5                          # no process group: identity
    assert list(rank_frames(1000, 100, 9, 16)) == list(range(900, 1000))
    assert list(rank_frames(1000, 100, 12, 16)) == list(range(200, 300))   # weak scaling wraps round the stream
