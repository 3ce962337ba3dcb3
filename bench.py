#!/usr/bin/env python
"""bench.py — ERI-derivative gradient throughput on synthetic water clusters (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A step = one pass of the whole hot path: tdg_set_system + tdg_plan + tdg_gradient on
the config-3 workload (256 waters, 6400 bf; the configuration BASELINE.json's target is quoted on).  Prints ONE JSON
line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
from paper_2407_16586_b200 import workload as wl  # noqa: E402

METRIC = "screened_quartets_per_s"
UNIT = "quartets/s"
ORACLE_SAMPLE_MOD = {0: 0, 1: 0, 2: 2000, 3: 20000, 4: 400000}
ORACLE_SEED = 7


def _workload_name(cfg):
    s = wl.CONFIGS[cfg]
    return "cfg%d: %d-water cluster, tau=%g, %s" % (cfg, s["waters"], s["tau"], "Schwarz x density" if s["density_weighted"] else "Schwarz")


def oracle_sample(cfg, sysm, mats, steps=1, warmup=0):
    """Times oracle.gradient on the deterministic subsample (S12); returns dict for cpu_baseline."""
    from oracle import oracle as orc

    orc.build()
    D, P, T = mats
    pairs, wJ, wK = wl.default_call(D, P, T)
    mod = ORACLE_SAMPLE_MOD[cfg]
    times, st = [], None
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        _, st = orc.gradient(sysm, pairs, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA, sample_mod=mod, sample_seed=ORACLE_SEED)
        if it >= warmup:
            times.append(time.perf_counter() - t0)
    dt = sum(times) / len(times)
    return dict(value=st["quartets_computed"] / dt, unit=UNIT, cores=orc.num_threads(), kind="oracle",
                sample="%s; canonical shell quartets with mix64 hash %% %d == 0 (seed %d): %d quartets in %.1f s (time includes the oracle's own "
                       "Schwarz bounds and screening loop)" % (_workload_name(cfg), mod, ORACLE_SEED, st["quartets_computed"], dt),
                seconds=dt, quartets=st["quartets_computed"])


class ClockSampler:
    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.QUERY, "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        # median over the busier half of the samples (idle gaps between steps pull the clock down)
        sm.sort()
        return dict(sm_mhz=statistics.median(sm[len(sm) // 2:]), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    sysm = wl.make_system(cfg)
    mats = wl.make_densities(sysm.nbf, wl.density_seed(cfg))
    r = oracle_sample(cfg, sysm, mats, steps=args.steps, warmup=min(args.warmup, 1))
    line = dict(impl="reference", metric=METRIC, value=r["value"], unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=min(args.warmup, 1),
                ms_per_step=r["seconds"] * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=_workload_name(cfg), nbf=sysm.nbf, natom=sysm.natom, note="CPU oracle on a bounded sample of the workload"),
                cpu_baseline=dict(value=r["value"], unit=UNIT, cores=r["cores"], kind="oracle", sample=r["sample"]),
                e2e=dict(value=r["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


def max_over_ranks(ms, dist, device):
    """Timing rule for N > 1: the step time is the MAX over ranks (replicas run independently, no data-path collective)."""
    if dist is None:
        return float(ms)
    import torch

    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, quartets_per_rank, ms):
    """Whole-job throughput: every rank processed `quartets_per_rank` quartets in `ms` (max over ranks)."""
    return world * quartets_per_rank / (ms * 1e-3)


def run_ours(args):
    import torch

    from paper_2407_16586_b200 import tdgrad

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    cfg = args.config
    ctx = tdgrad.Context(local)
    shard = args.parallelism == "shard" and world > 1      # work items dealt over ranks + one all-reduce
    if shard:
        ctx.set_shard(rank, world)
    peak_tf = ctx.fp64_peak(400.0)
    sysm = wl.make_system(cfg)
    nbf, natom = sysm.nbf, sysm.natom
    D, P, T = wl.make_densities_torch(nbf, 20240716 + cfg, dev)
    pairs, wJ, wK = wl.default_call(D, P, T)
    g_dev = torch.zeros((natom, 3), dtype=torch.float64, device=dev)

    def step(mats, out, stats=True):
        ctx.set_system(sysm)                                   # a0
        ctx.plan(sysm.tau, sysm.density_weighted, 0, 0)       # a1-a2 (Schwarz on device, sort, work lists)
        g, st = ctx.gradient(mats, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA, stream=torch.cuda.current_stream().cuda_stream,
                             out=out, want_stats=stats)      # a3-a9
        if shard:                                              # the path's one exchange step: 3*natom doubles over NCCL
            g = tdgrad.allreduce_partial(g if out is not None else torch.from_numpy(g).to(dev))
            if out is None:
                g = g.cpu().numpy()
        return g, st

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(pairs, g_dev)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    agg_ms, agg_q, agg_p = [0.0] * tdgrad.NCLASS, [0] * tdgrad.NCLASS, [0] * tdgrad.NCLASS
    launches, quartets = 0, 0
    e0.record()
    for _ in range(args.steps):
        _, st = step(pairs, g_dev)
        launches += st["launches"] + 1     # + the Schwarz kernel of tdg_plan
        quartets += st["quartets_computed"]
        for c in range(tdgrad.NCLASS):
            agg_ms[c] += st["ms_by_class"][c]; agg_q[c] += st["quartets_by_class"][c]; agg_p[c] += st["prim_quartets_by_class"][c]
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    ms = max_over_ranks(ms, dist, dev)
    g_host = g_dev.cpu().numpy()
    total_quartets = quartets
    if shard:   # every rank computed its own share of the quartets
        tq = torch.tensor([quartets], dtype=torch.int64, device=dev)
        dist.all_reduce(tq, op=dist.ReduceOp.SUM)
        total_quartets = int(tq.item())
    # end-to-end through the C ABI with HOST buffers (pinned), copies inside the timed region; rank 0 alone for replicas,
    # every rank (partial gradients all-reduced, max over ranks) when the work is sharded
    e2e_dt = None
    if rank == 0 or shard:
        hD, hP, hT = [x.cpu().pin_memory().numpy() for x in (D, P, T)]
        hpairs, _, _ = wl.default_call(hD, hP, hT)
        e2e_warm = 0 if ms / args.steps > 20000 else 1
        for _ in range(e2e_warm):
            step(hpairs, None, stats=False)
        if shard:
            barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        g2, _ = step(hpairs, None, stats=False)
        torch.cuda.synchronize()
        e2e_dt = time.perf_counter() - t0
        if shard:
            e2e_dt = max_over_ranks(e2e_dt, dist, dev)
        assert np.max(np.abs(g2 - g_host)) < 1e-8, "host-buffer and device-buffer paths disagree"
    if rank == 0:
        value = aggregate_value(1, total_quartets, ms) if shard else aggregate_value(world, quartets, ms)
        # roofline of the dominant class kernel (largest share of the step)
        top = max(range(tdgrad.NCLASS), key=lambda c: agg_ms[c])
        fl_top = tdgrad.model_flops(top, agg_q[top], agg_p[top])
        fl_all = sum(tdgrad.model_flops(c, agg_q[c], agg_p[c]) for c in range(tdgrad.NCLASS))
        achieved = fl_top / (agg_ms[top] * 1e-3) * 1e-12
        traffic, executed = None, {}
        tpath = os.path.join(ROOT, "profiles", "traffic.json")   # numbers read off the committed ncu captures (data only)
        if os.path.exists(tpath):
            rec = json.load(open(tpath)).get(tdgrad.class_name(top))
            if rec:
                traffic = rec.get("dram_bytes")
                executed = dict(executed_tflops=rec.get("executed_tflops"), executed_frac=rec.get("executed_tflops", 0.0) / peak_tf,
                                fp64_pipe_pct=rec.get("fp64_pipe_pct"),
                                executed_note="FP64 FLOPs actually executed (ncu: 2*DFMA+DMUL+DADD) by the largest launch of this kernel, "
                                              "profiles/r01_ncu_full_*.md; `achieved` uses SURVEY.md 8(d)'s algorithmic model, which charges 2-4x more")
        roofline = dict(bound="alu", achieved=achieved, peak=peak_tf, unit="TFLOP/s", frac=achieved / peak_tf, traffic=traffic, **executed,
                        kernel="tdg_grad_kernel" + tdgrad.class_name(top), kernel_share_of_step=agg_ms[top] / ms,
                        peak_source="FP64 FMA-chain microbenchmark run live on this GPU (tdg_fp64_peak); nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
                        whole_step_model_tflops=fl_all / (ms * 1e-3) * 1e-12, whole_step_frac=fl_all / (ms * 1e-3) * 1e-12 / peak_tf)
        dt = e2e_dt
        h2d = 3 * nbf * nbf * 8 + sysm.xyz.nbytes + sysm.exps.nbytes + sysm.coefs.nbytes + sysm.shells.nbytes
        e2e = dict(value=((total_quartets if shard else quartets) / args.steps) / dt, unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(natom * 3 * 8), seconds=dt)
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            cpu = oracle_sample(cfg, sysm, (hD, hP, hT))
            cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}
        per_class = {tdgrad.class_name(c): dict(quartets=agg_q[c] // args.steps, ms=agg_ms[c] / args.steps,
                                               model_tflops=tdgrad.model_flops(c, agg_q[c], agg_p[c]) / (agg_ms[c] * 1e-3) * 1e-12)
                     for c in range(tdgrad.NCLASS) if agg_q[c]}
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=ms / args.steps,
                    higher_is_better=True, scaling="strong" if shard else "weak", vs_baseline=None, dtype="f64", data="synthetic",
                    config=dict(workload=_workload_name(cfg), nbf=nbf, natom=natom, nshell=sysm.nshell, pairs=3, omega=wl.OMEGA,
                                l2="inputs (3 x %.0f MB densities) larger than L2" % (nbf * nbf * 8 / 1e6),
                                parallelism=("shard%d+allreduce" % world) if shard else ("replicas" if world > 1 else "1gpu")),
                    wall_time_s=ms / args.steps * 1e-3, quartets_per_step=total_quartets // args.steps,
                    grad_sum_abs_max=float(np.max(np.abs(g_host.sum(axis=0)))),
                    roofline=roofline, cpu_baseline=cpu, e2e=e2e, gpu_launches=launches, clocks=clocks, per_class=per_class)
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "shard"],
                    help="N > 1: independent replicas (weak scaling, default) or work items sharded over ranks + one NCCL all-reduce (strong)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
