"""One tdg_gradient call on a BASELINE.json config, for use under ncu (profiles/*.md name the full commands).

    python -m paper_2407_16586_b200.profile_run [config=3] [calls=1]
"""
import sys

import torch

from paper_2407_16586_b200 import tdgrad
from paper_2407_16586_b200 import workload as wl


def main():
    cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 3
    calls = int(sys.argv[2]) if len(sys.argv) > 2 else 1
    ctx = tdgrad.Context(0)
    s = wl.make_system(cfg)
    ctx.set_system(s)
    ctx.plan(s.tau, s.density_weighted)
    D, P, T = wl.make_densities_torch(s.nbf, 20240716 + cfg, "cuda")
    pairs, wJ, wK = wl.default_call(D, P, T)
    for _ in range(calls):
        g, st = ctx.gradient(pairs, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA)
    print("quartets", st["quartets_computed"], "ms", st["ms_total"])
    ctx.close()


if __name__ == "__main__":
    main()
