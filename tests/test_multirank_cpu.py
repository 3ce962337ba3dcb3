"""N > 1 path on CPU: two gloo ranks, max-over-ranks timing and whole-job aggregation of bench.py, and the one
exchange step of the sharded path (sum of the per-rank partial gradients)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(100.0 + 50.0 * rank, dist, torch.device("cpu"))
    dist.barrier()
    if rank == 0:
        out.put((ms, bench.aggregate_value(world, 1000, ms)))
    dist.destroy_process_group()


def test_two_rank_timing_and_aggregation():
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    ms, value = q.get()
    assert ms == 150.0
    assert abs(value - 2 * 1000 / 0.150) < 1e-9


def _allreduce_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    from paper_2407_16586_b200 import tdgrad

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    assert tdgrad.shard_of_env() == (rank, world)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    natom = 5
    full = torch.arange(3 * natom, dtype=torch.float64).reshape(natom, 3) / 7.0
    partial = torch.zeros_like(full)
    partial.view(-1)[rank::world] = full.view(-1)[rank::world]     # this rank's share of the contributions
    g = tdgrad.allreduce_partial(partial)
    ok = bool(torch.equal(g, full)) and g.data_ptr() == partial.data_ptr()
    flags = [None] * world
    dist.all_gather_object(flags, ok)
    if rank == 0:
        out.put(all(flags))
    dist.destroy_process_group()


def test_two_rank_partial_gradient_allreduce():
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_allreduce_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert q.get() is True


def test_allreduce_partial_without_process_group_is_identity():
    sys.path.insert(0, ROOT)
    from paper_2407_16586_b200 import tdgrad

    t = torch.ones(4, 3, dtype=torch.float64)
    assert tdgrad.allreduce_partial(t) is t and tdgrad.shard_of_env() == (0, 1)


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.max_over_ranks(12.5, None, None) == 12.5
