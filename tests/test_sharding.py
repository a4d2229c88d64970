"""N > 1 path (replicas only) on CPU: world_size-2 gloo run of the rank -> event-seed
assignment and the max-over-ranks timing reduction that bench.py uses."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2209_13711_b200 import sharding as S


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, per_rank, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seeds = S.event_seeds(rank, world, per_rank)
    gathered = [None] * world
    dist.all_gather_object(gathered, seeds)
    ms = S.max_over_ranks(10.0 + 5.0 * rank, dist)          # rank 1 is the slow one
    dist.barrier()
    if rank == 0:
        out.put((gathered, ms))
    dist.destroy_process_group()


def test_two_rank_event_sharding_and_timing():
    world, per_rank = 2, 64
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, per_rank, out)) for r in range(world)]
    for p in procs:
        p.start()
    gathered, ms = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    flat = [s for g in gathered for s in g]
    assert len(flat) == world * per_rank and len(set(flat)) == len(flat)      # disjoint
    assert sorted(flat) == list(range(S.BASE_SEED, S.BASE_SEED + world * per_rank))
    assert gathered[0] == S.event_seeds(0, 1, per_rank)                        # rank 0 = the 1-GPU workload
    assert ms == 15.0                                                           # max over ranks
    assert S.job_events_per_s(world, per_rank, 3, ms) == world * per_rank * 3 / 0.015


def test_single_process_is_identity():
    assert S.max_over_ranks(7.5) == 7.5
    assert S.event_seeds(0, 1, 3) == [1000, 1001, 1002]
