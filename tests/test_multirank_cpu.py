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


class _StubContext:
    """Stands in for tdgrad.Context on CPU: every rank returns its share of a fixed 'gradient' and of the quartets, so the
    test can check bench.run_ours's N > 1 logic (sharding call, all-reduce, max-over-ranks time, whole-job aggregation)."""

    def __init__(self, natom, log):
        self.natom, self.log, self.rank, self.n = natom, log, 0, 1

    def set_shard(self, rank, n):
        self.rank, self.n = rank, n
        self.log.append(("set_shard", rank, n))

    def set_streams(self, n):
        pass

    def fp64_peak(self, ms):
        return 30.0

    def set_system(self, s):
        pass

    def plan(self, *a):
        pass

    def gradient(self, mats, wJ, wK, cJ, cK, cLR, omega, stream=None, out=None, want_stats=True):
        import numpy as np

        full = np.arange(3 * self.natom, dtype=np.float64).reshape(self.natom, 3)
        part = np.zeros_like(full)
        part.reshape(-1)[self.rank::self.n] = full.reshape(-1)[self.rank::self.n]
        if out is not None:
            out.copy_(torch.from_numpy(part))
            g = out
        else:
            g = part
        st = None
        if want_stats:
            q = [0] * 55
            q[1] = 1000 + 100 * self.rank           # ranks own different numbers of quartets
            ms = [0.0] * 55
            ms[1] = 5.0
            st = dict(launches=3, quartets_computed=q[1], quartets_by_class=q, prim_quartets_by_class=q, ms_by_class=ms)
        return g, st

    def close(self):
        pass


class _StubBackend:
    dist_backend = "gloo"

    def __init__(self, natom, rank):
        from paper_2407_16586_b200 import tdgrad

        self.tdgrad, self.device, self.natom, self.rank, self.log = tdgrad, torch.device("cpu"), natom, rank, []

    def context(self):
        return _StubContext(self.natom, self.log)

    def densities(self, nbf, seed, sysm=None, kind="dense"):
        return [torch.zeros(2, 2, dtype=torch.float64) for _ in range(3)]

    def host_copies(self, mats):
        return [m.numpy() for m in mats]

    def stream(self):
        return 0

    def synchronize(self):
        pass

    def timer(self):
        import time

        return time.perf_counter()

    def elapsed_ms(self, e0, e1):
        return 100.0 + 40.0 * self.rank             # rank 1 is the slow one

    def clock_sampler(self):
        class S:
            def stop(self):
                return dict(sm_mhz=None, sm_max_mhz=None, reasons=["stub"])
        return S()


def _bench_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import argparse
    import json

    import bench
    from paper_2407_16586_b200 import workload as wl

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    args = argparse.Namespace(gpus=world, steps=2, warmup=1, config=0, parallelism="shard", streams=1, densities="dense", no_cpu_baseline=True)
    be = _StubBackend(wl.make_system(0).natom, rank)
    lines = []
    bench.run_ours(args, backend=be, emit=lines.append)
    if rank == 0:
        out.put((json.loads(lines[0]), be.log))
    else:
        assert not lines                               # only rank 0 prints
    dist.barrier()
    dist.destroy_process_group()


def test_bench_shard_branch_end_to_end_on_two_gloo_ranks():
    """bench.run_ours with WORLD_SIZE=2 and the default --parallelism: set_shard(rank, 2) on every rank, partial gradients
    all-reduced, time = max over ranks, value = quartets of ALL ranks / that time, "scaling": "strong"."""
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_bench_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(180)
        assert p.exitcode == 0
    line, log = q.get()
    assert ("set_shard", 0, 2) in log
    assert line["scaling"] == "strong" and line["n_gpus"] == 2
    assert line["config"]["parallelism"] == "shard2+allreduce"
    assert line["ms_per_step"] == 140.0 / 2                      # max over ranks of (100, 140) ms for 2 steps
    total_q = 2 * (1000 + 1100)                                  # both ranks, both steps
    assert line["quartets_per_step"] == total_q // 2
    assert abs(line["value"] - total_q / 0.140) < 1e-6
    assert line["grad_sum_abs_max"] > 0                          # the all-reduced gradient is the full one
    assert line["e2e"]["value"] > 0 and line["gpu_launches"] == 2 * 4


def test_bench_defaults_to_sharding_for_n_gt_1():
    sys.path.insert(0, ROOT)
    import bench

    old = sys.argv
    try:
        sys.argv = ["bench.py", "--gpus", "8"]
        import argparse

        ap_args = None

        def fake_run(args, **kw):
            nonlocal ap_args
            ap_args = args
        orig = bench.run_ours
        bench.run_ours = fake_run
        bench.main()
        bench.run_ours = orig
    finally:
        sys.argv = old
    assert ap_args.parallelism == "shard"
