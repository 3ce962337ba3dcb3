"""One tdg_gradient call on a BASELINE.json config, for use under ncu (profiles/*.md name the full commands).

    python -m paper_2407_16586_b200.profile_run [config=3] [calls=1] [dense|decaying]
"""
import json
import os
import sys

import torch

from paper_2407_16586_b200 import ncu_classes, tdgrad
from paper_2407_16586_b200 import workload as wl


def main():
    cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 3
    calls = int(sys.argv[2]) if len(sys.argv) > 2 else 1
    ctx = tdgrad.Context(0)
    s = wl.make_system(cfg)
    ctx.set_system(s)
    ctx.plan(s.tau, s.density_weighted)
    kind = sys.argv[3] if len(sys.argv) > 3 else "dense"
    D, P, T = (wl.make_decaying_densities_torch(s, 20240716 + cfg, "cuda") if kind == "decaying"
               else wl.make_densities_torch(s.nbf, 20240716 + cfg, "cuda"))
    pairs, wJ, wK = wl.default_call(D, P, T)
    for _ in range(calls):
        g, st = ctx.gradient(pairs, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA)
    print("quartets", st["quartets_computed"], "ms", st["ms_total"])
    os.makedirs("gpurun_out", exist_ok=True)    # per-class counts of the profiled call, merged into the summary by ncu_classes.py
    with open(os.path.join("gpurun_out", "profile_run_cfg%d.json" % cfg), "w") as fh:
        json.dump(dict(config=cfg, source_hash=ncu_classes.source_hash(), quartets=st["quartets_computed"], ms_total=st["ms_total"],
                       quartets_by_class={tdgrad.class_name(c): st["quartets_by_class"][c] for c in range(tdgrad.NCLASS) if st["quartets_by_class"][c]},
                       prim_quartets_by_class={tdgrad.class_name(c): st["prim_quartets_by_class"][c] for c in range(tdgrad.NCLASS) if st["quartets_by_class"][c]},
                       ms_by_class={tdgrad.class_name(c): st["ms_by_class"][c] for c in range(tdgrad.NCLASS) if st["quartets_by_class"][c]}), fh)
    ctx.close()


if __name__ == "__main__":
    main()
