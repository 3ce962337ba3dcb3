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
ORACLE_SAMPLE_MOD = {0: 0, 1: 0, 2: 300, 3: 8000, 4: 400000}   # sized for ~20-40 s of oracle integrals on a 16-core host
ORACLE_SEED = 7


def _workload_name(cfg):
    s = wl.CONFIGS[cfg]
    return "cfg%d: %d-water cluster, tau=%g, %s" % (cfg, s["waters"], s["tau"], "Schwarz x density" if s["density_weighted"] else "Schwarz")


def oracle_sample(cfg, sysm, mats, steps=1, warmup=0):
    """Times the CPU oracle (as it stands: plain C, gcc -O2, OpenMP) on the deterministic subsample (S12) of the workload.

    Two phases are timed apart, because at cfg 3-4 the oracle's own Schwarz bounds and O(pairs^2) screening loop cost as
    much as its integrals: `seconds_screening` is a pass whose subsample keeps no quartet (Schwarz + density maxima +
    screening loop only), `seconds_integrals` = full pass - that.  `value` = sampled quartets / seconds_integrals: the
    oracle's throughput on the work the GPU metric counts.  An unoptimised checker, not a tuned CPU code: a baseline, not a target."""
    from oracle import oracle as orc

    orc.build()
    D, P, T = mats
    pairs, wJ, wK = wl.default_call(D, P, T)
    mod = ORACLE_SAMPLE_MOD[cfg]
    args = (sysm, pairs, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA)
    t0 = time.perf_counter()
    _, st0 = orc.gradient(*args, sample_mod=0xFFFFFFFB, sample_seed=ORACLE_SEED)      # keeps (almost surely) no quartet
    t_screen = time.perf_counter() - t0
    times, st = [], None
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        _, st = orc.gradient(*args, sample_mod=mod, sample_seed=ORACLE_SEED)
        if it >= warmup:
            times.append(time.perf_counter() - t0)
    dt = sum(times) / len(times)
    nq = st["quartets_computed"] - st0["quartets_computed"]
    t_int = max(dt - t_screen, 1e-9)
    return dict(value=nq / t_int, unit=UNIT, cores=orc.num_threads(), kind="oracle",
                sample="%s; canonical shell quartets with mix64 hash %% %d == 0 (seed %d): %d quartets; oracle pass %.1f s = %.1f s Schwarz bounds + "
                       "screening loop over all pairs (timed apart, sample that keeps nothing) + %.1f s integrals and contraction; value = quartets / "
                       "integral seconds" % (_workload_name(cfg), mod, ORACLE_SEED, nq, dt, t_screen, t_int),
                seconds=dt, seconds_screening=t_screen, seconds_integrals=t_int, quartets=nq)


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


def _config(cfg, sysm, parallelism):
    nbf = sysm.nbf
    return dict(workload=_workload_name(cfg), nbf=nbf, natom=sysm.natom, nshell=sysm.nshell, pairs=3, omega=wl.OMEGA,
                l2="inputs (3 x %.0f MB densities) larger than L2" % (nbf * nbf * 8 / 1e6), parallelism=parallelism)


def run_reference(args):
    """Reference arm = the CPU oracle as it stands, on the box's host cores (rank 0 only).  A step = one oracle pass over a
    bounded deterministic subsample of the same workload; with many steps the sample is the small one (the oracle's
    Schwarz + screening phase alone costs ~20 s per pass at cfg 3, so the run is bounded by the number of passes)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    if args.steps + args.warmup > 4:
        ORACLE_SAMPLE_MOD[3] = max(ORACLE_SAMPLE_MOD[3], 20000)
    warm = min(args.warmup, 1)
    sysm = wl.make_system(cfg)
    mats = wl.make_densities(sysm.nbf, wl.density_seed(cfg))
    r = oracle_sample(cfg, sysm, mats, steps=args.steps, warmup=warm)
    value = r["quartets"] / r["seconds"]           # whole pass (screening included): consistent with ms_per_step
    line = dict(impl="reference", metric=METRIC, value=value, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=warm,
                ms_per_step=r["seconds"] * 1e3, higher_is_better=True, scaling="strong" if args.gpus > 1 else "weak", vs_baseline=None, dtype="f64",
                data="synthetic", config=_config(cfg, sysm, "cpu-oracle"),
                cpu_baseline=dict(value=value, unit=UNIT, cores=r["cores"], kind="oracle", sample=r["sample"], seconds_screening=r["seconds_screening"],
                                  seconds_integrals=r["seconds_integrals"], value_integral_phase_only=r["value"],
                                  note="unoptimised checker (plain C, gcc -O2), not a tuned CPU implementation: the ratio to it is not a speedup claim"),
                e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
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


def roofline_of(agg_ms, agg_q, agg_p, step_ms, peak_tf, cfg, nsteps):
    """Roofline object of the bench line for the dominant class kernel (largest share of the step).

    achieved = FP64 FLOPs the kernel EXECUTES on this workload (ncu thread-level counts 2*DFMA + DMUL + DADD, summed over the
    class's launches; profiles/r02_ncu_classes_cfg<N>.json, captured with the command named in the .md beside it) divided by the
    kernel's device time in THIS run (CUDA events around every launch, tdg_stats).  The capture is tied to the kernel sources
    by a hash; when the sources changed since, or the quartet counts differ, the executed numbers are null rather than stale.
    `model_*` = the algorithmic FLOP model of SURVEY.md 8(d), which charges several times more than the kernels execute."""
    from paper_2407_16586_b200 import ncu_classes, tdgrad

    top = max(range(tdgrad.NCLASS), key=lambda c: agg_ms[c])
    name = tdgrad.class_name(top)
    sec = agg_ms[top] * 1e-3
    model_top = tdgrad.model_flops(top, agg_q[top], agg_p[top]) / sec * 1e-12
    model_all = sum(tdgrad.model_flops(c, agg_q[c], agg_p[c]) for c in range(tdgrad.NCLASS)) / (step_ms * 1e-3) * 1e-12
    out = dict(bound="alu", achieved=None, peak=peak_tf, unit="TFLOP/s", frac=None, traffic=None, kernel="tdg_grad_kernel" + name,
               kernel_share_of_step=agg_ms[top] / step_ms,
               peak_source="FP64 FMA-chain microbenchmark run live on this GPU (tdg_fp64_peak; MEASURED_PEAKS.json has no FP64 entry); nominal "
                           "148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
               model_tflops=model_top, model_frac=model_top / peak_tf, whole_step_model_tflops=model_all)
    path = os.path.join(ROOT, "profiles", "r02_ncu_classes_cfg%d.json" % cfg)
    note = None
    if not os.path.exists(path):
        note = "no ncu capture for this config under profiles/"
    else:
        rec = json.load(open(path))
        if rec.get("source_hash") != ncu_classes.source_hash():
            note = "ncu capture %s is older than the kernel sources (hash %s != %s): executed FLOPs not reported" % (
                os.path.basename(path), rec.get("source_hash"), ncu_classes.source_hash())
        else:
            steps = nsteps
            cl = rec["classes"]
            c = cl.get(name)
            qcap = rec.get("quartets_by_class", {}).get(name)
            if qcap is not None and qcap * steps != agg_q[top]:
                note = "ncu capture was taken on a different workload (%d quartets of %s per call, this run %d)" % (qcap, name, agg_q[top] // steps)
            elif c:
                out.update(achieved=c["flops"] * steps / sec * 1e-12, traffic=(c["dram_read"] + c["dram_write"]),
                           fp64_pipe_pct_under_ncu=c["fp64_pipe_pct"], warps_active_pct_under_ncu=c["warps_active_pct"], registers=c["regs"],
                           executed_flop_per_quartet=c["flops"] * steps / agg_q[top], capture=os.path.basename(path), capture_hash=rec["source_hash"])
                out["frac"] = out["achieved"] / peak_tf
                done = [(tdgrad.class_name(k), agg_ms[k]) for k in range(tdgrad.NCLASS) if agg_q[k]]
                fl = sum(cl[nm]["flops"] for nm, _ in done if nm in cl) * steps
                out["whole_step_executed_tflops"] = fl / (step_ms * 1e-3) * 1e-12
                out["whole_step_frac"] = out["whole_step_executed_tflops"] / peak_tf
                out["per_class_executed_frac"] = {nm: round(cl[nm]["flops"] * steps / (t * 1e-3) * 1e-12 / peak_tf, 4) for nm, t in done if nm in cl and t > 0}
    if note:
        out["note"] = note
    return out


class CudaBackend:
    """Everything run_ours needs from the machine: the CUDA library binding, device tensors, device timing, the process group.
    tests/test_multirank_cpu.py substitutes a CPU stub with the same methods to drive the N > 1 logic under gloo."""

    dist_backend = "nccl"

    def __init__(self, local):
        import torch

        from paper_2407_16586_b200 import tdgrad

        if not torch.cuda.is_available():
            raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
        torch.cuda.set_device(local)
        self.torch, self.tdgrad, self.local = torch, tdgrad, local
        self.device = torch.device("cuda", local)

    def context(self):
        return self.tdgrad.Context(self.local)

    def densities(self, nbf, seed, sysm=None, kind="dense"):
        if kind == "decaying":     # spatially decaying densities (workload.make_decaying_densities_torch)
            return wl.make_decaying_densities_torch(sysm, seed, self.device)
        return wl.make_densities_torch(nbf, seed, self.device)

    def host_copies(self, mats):
        return [x.cpu().pin_memory().numpy() for x in mats]

    def stream(self):
        return self.torch.cuda.current_stream().cuda_stream

    def synchronize(self):
        self.torch.cuda.synchronize()

    def timer(self):
        e = self.torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    def elapsed_ms(self, e0, e1):
        return e0.elapsed_time(e1)

    def clock_sampler(self):
        return ClockSampler(self.local)


def run_ours(args, backend=None, emit=print):
    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    be = backend if backend is not None else CudaBackend(local)
    tdgrad = be.tdgrad
    dev = be.device
    dist = None
    if world > 1:
        import torch.distributed as dist

        if not dist.is_initialized():
            dist.init_process_group(be.dist_backend, **(dict(device_id=dev) if be.dist_backend == "nccl" else {}))
    cfg = args.config
    ctx = be.context()
    # for N > 1 the work items are dealt over the ranks and the partial gradients all-reduced (strong scaling);
    # independent replicas only on request
    shard = world > 1 and args.parallelism != "replicas"
    if shard:
        ctx.set_shard(rank, world)
    if args.streams > 1:
        ctx.set_streams(args.streams)
    peak_tf = ctx.fp64_peak(400.0)
    sysm = wl.make_system(cfg)
    nbf, natom = sysm.nbf, sysm.natom
    D, P, T = be.densities(nbf, 20240716 + cfg, sysm, args.densities)
    pairs, wJ, wK = wl.default_call(D, P, T)
    g_dev = torch.zeros((natom, 3), dtype=torch.float64, device=dev)

    def step(mats, out, stats=True):
        ctx.set_system(sysm)                                   # a0
        ctx.plan(sysm.tau, sysm.density_weighted, 0, 0)       # a1-a2 (Schwarz on device, sort, work lists)
        g, st = ctx.gradient(mats, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA, stream=be.stream(), out=out, want_stats=stats)      # a3-a9
        if shard:                                              # the path's one exchange step: 3*natom doubles over NCCL
            g = tdgrad.allreduce_partial(g if out is not None else torch.from_numpy(g).to(dev))
            if out is None:
                g = g.cpu().numpy()
        return g, st

    def barrier():
        if dist is not None:
            dist.barrier()
        be.synchronize()

    probe = None
    for _ in range(args.warmup):
        _, probe = step(pairs, g_dev)
    if shard and probe is None:
        _, probe = step(pairs, g_dev)
    barrier()
    sampler = be.clock_sampler() if rank == 0 else None
    agg_ms, agg_q, agg_p = [0.0] * tdgrad.NCLASS, [0] * tdgrad.NCLASS, [0] * tdgrad.NCLASS
    launches, quartets = 0, 0
    roof_steps = args.steps

    def add(st):
        for c in range(tdgrad.NCLASS):
            agg_ms[c] += st["ms_by_class"][c]; agg_q[c] += st["quartets_by_class"][c]; agg_p[c] += st["prim_quartets_by_class"][c]

    e0 = be.timer()
    for _ in range(args.steps):
        if shard:
            # sharded steps run WITHOUT per-class event timing: the class launches then free-run over the streams and the tail of one
            # class overlaps the next (csrc/tdg_api.cu launch_classes).  Quartet and launch counts are those of the instrumented
            # warm-up call on the same inputs and plan (deterministic).
            step(pairs, g_dev, stats=False)
            st = probe
        else:
            _, st = step(pairs, g_dev)
            add(st)
        launches += st["launches"] + 1     # + the Schwarz kernel of tdg_plan
        quartets += st["quartets_computed"]
    e1 = be.timer()
    barrier()
    if shard:
        add(probe)
        roof_steps = 1
    ms = be.elapsed_ms(e0, e1)
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
    if (rank == 0 or shard) and not getattr(args, "no_e2e", False):
        hD, hP, hT = be.host_copies((D, P, T))
        hpairs, _, _ = wl.default_call(hD, hP, hT)
        e2e_warm = 0 if ms / args.steps > 20000 else 1
        for _ in range(e2e_warm):
            step(hpairs, None, stats=False)
        if shard:
            barrier()
        be.synchronize()
        t0 = time.perf_counter()
        g2, _ = step(hpairs, None, stats=False)
        be.synchronize()
        e2e_dt = time.perf_counter() - t0
        if shard:
            e2e_dt = max_over_ranks(e2e_dt, dist, dev)
        assert np.max(np.abs(g2 - g_host)) < 1e-8, "host-buffer and device-buffer paths disagree"
    if rank == 0:
        value = aggregate_value(1, total_quartets, ms) if shard else aggregate_value(world, quartets, ms)
        roofline = roofline_of(agg_ms, agg_q, agg_p, ms if not shard else ms / args.steps, peak_tf, cfg, roof_steps)
        dt = e2e_dt
        h2d = 3 * nbf * nbf * 8 + sysm.xyz.nbytes + sysm.exps.nbytes + sysm.coefs.nbytes + sysm.shells.nbytes
        e2e = None if dt is None else dict(value=((total_quartets if shard else quartets) / args.steps) / dt, unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(natom * 3 * 8), seconds=dt)
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            if e2e_dt is None:
                hD, hP, hT = be.host_copies((D, P, T))
            cpu = oracle_sample(cfg, sysm, (hD, hP, hT))
            cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "seconds_screening", "seconds_integrals")}
            cpu["note"] = "unoptimised checker (plain C, gcc -O2), not a tuned CPU implementation: the ratio to it is not a speedup claim"
        per_class = {tdgrad.class_name(c): dict(quartets=agg_q[c] // roof_steps, ms=agg_ms[c] / roof_steps,
                                               model_tflops=tdgrad.model_flops(c, agg_q[c], agg_p[c]) / (agg_ms[c] * 1e-3) * 1e-12)
                     for c in range(tdgrad.NCLASS) if agg_q[c] and agg_ms[c] > 0}
        config = _config(cfg, sysm, ("shard%d+allreduce" % world) if shard else ("replicas" if world > 1 else "1gpu"))
        config["streams"] = args.streams
        config["per_class_timing"] = ("instrumented warm-up call of rank 0 (timed steps free-run the class launches over the streams)" if shard
                                      else "CUDA events around every class inside the timed steps")
        config["densities"] = args.densities
        if args.densities != "dense":
            config["workload"] += "; densities decaying as exp(-r / %.1f bohr) (workload.make_decaying_densities)" % wl.DECAY_LENGTH
        line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=ms / args.steps,
                    higher_is_better=True, scaling="strong" if shard else "weak", vs_baseline=None, dtype="f64", data="synthetic",
                    config=config, wall_time_s=ms / args.steps * 1e-3, quartets_per_step=total_quartets // args.steps,
                    grad_sum_abs_max=float(np.max(np.abs(g_host.sum(axis=0)))),
                    roofline=roofline, cpu_baseline=cpu, e2e=e2e, gpu_launches=launches, clocks=clocks, per_class=per_class)
        emit(json.dumps(line))
    if dist is not None and backend is None:
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
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg (profiling runs under ncu; `e2e` is then null)")
    ap.add_argument("--densities", default="dense", choices=["dense", "decaying"],
                    help="dense: BASELINE.json's random matrices; decaying: second workload with spatially decaying densities (NEXT-4)")
    ap.add_argument("--streams", type=int, default=1, help="CUDA streams the class launches of a call are dealt over (tdg_set_streams)")
    ap.add_argument("--parallelism", default="shard", choices=["shard", "replicas"],
                    help="N > 1: work items sharded over the ranks + one NCCL all-reduce of the gradient (strong scaling, default), or independent replicas")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
