"""Load balance of the rank shards (tdg_set_shard) measured on ONE GPU: for each world size N the N
shards run one after another, each to completion (no rank waits on another), and the device time of each is recorded.
The predicted N-GPU step is the slowest shard; efficiency = unsharded time / (N x slowest shard).  The all-reduce of
3*natom doubles (18 KB at cfg 3) is not in these numbers.

    python -m paper_2407_16586_b200.shard_balance [config=3] [world sizes=2,4,8]
"""
import json
import sys

import numpy as np
import torch

from paper_2407_16586_b200 import tdgrad
from paper_2407_16586_b200 import workload as wl


def main():
    cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 3
    worlds = [int(x) for x in (sys.argv[2] if len(sys.argv) > 2 else "2,4,8").split(",")]
    ctx = tdgrad.Context(0)
    s = wl.make_system(cfg)
    ctx.set_system(s)
    D, P, T = wl.make_densities_torch(s.nbf, 20240716 + cfg, "cuda")
    pairs, wJ, wK = wl.default_call(D, P, T)

    def run(rank, n):
        """One shard: an instrumented call (counts, gradient), then the call as bench.py's timed steps make it (no per-class event
        timing, so the class launches of a shard free-run over the streams), timed with CUDA events on the launching stream."""
        ctx.set_shard(rank, n)
        ctx.plan(s.tau, s.density_weighted)
        g, st = ctx.gradient(pairs, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA)
        out = torch.zeros((s.natom, 3), dtype=torch.float64, device="cuda")
        best = None
        for _ in range(2):      # best of 2: a single call shows outliers of ~10 % now and then
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.gradient(pairs, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA, out=out, want_stats=False)
            e1.record()
            torch.cuda.synchronize()
            best = e0.elapsed_time(e1) if best is None else min(best, e0.elapsed_time(e1))
        st["ms_instrumented"] = st["ms_total"]
        st["ms_total"] = best
        return g, st

    run(0, 1)                      # warm-up
    g1, st1 = run(0, 1)
    out = dict(config=cfg, unsharded_ms=st1["ms_total"], quartets=st1["quartets_computed"], worlds=[])
    for n in worlds:
        ms, ms_i, q, total = [], [], [], np.zeros_like(g1)
        for r in range(n):
            g, st = run(r, n)
            ms.append(st["ms_total"]); q.append(st["quartets_computed"]); total += g; ms_i.append(st["ms_instrumented"])
        assert sum(q) == st1["quartets_computed"]
        out["worlds"].append(dict(n=n, shard_ms=ms, shard_ms_with_per_class_timing=ms_i, shard_quartets=q, slowest_ms=max(ms), efficiency=st1["ms_total"] / (n * max(ms)),
                                  max_abs_diff_vs_unsharded=float(np.max(np.abs(total - g1)))))
    print(json.dumps(out))
    ctx.close()


if __name__ == "__main__":
    main()
