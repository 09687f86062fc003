"""world_size-2 gloo test (CPU) of the multi-rank host logic bench.py uses: frame sharding without overlap, max-over-ranks
timing, summed unit counts (tier framing 5: the path shards by frame set with no data-path collective)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1809_06132_b200 import shard


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    frames = shard.frames_for_rank(0, 32, rank, world)
    strong = shard.split_stream(33, rank, world)
    ms, units = shard.reduce_timing([10.0 + 5.0 * rank, 3.0 - rank], [float(len(frames)) * 1000.0])
    gathered = [None] * world
    dist.all_gather_object(gathered, (frames, strong))
    dist.barrier()
    if rank == 0:
        out.put((ms, units, gathered))
    dist.destroy_process_group()


def test_two_rank_sharding_and_timing_reduce():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    ms, units, gathered = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == [15.0, 3.0]                 # max over ranks
    assert units == [64000.0]                # summed over ranks
    weak = [f for fr, _ in gathered for f in fr]
    assert sorted(weak) == list(range(64)) and len(set(weak)) == 64
    strong = [f for _, st in gathered for f in st]
    assert strong == list(range(33))
    assert abs(len(gathered[0][1]) - len(gathered[1][1])) <= 1


def test_single_process_is_identity():
    ms, units = shard.reduce_timing([1.5], [7.0])
    assert ms == [1.5] and units == [7.0]
    assert shard.frames_for_rank(5, 4, 0, 1) == [5, 6, 7, 8]
    assert shard.split_stream(5, 0, 1) == [0, 1, 2, 3, 4]
