"""Writes tests/golden/cfg0_gradient.txt by calling ONLY the CPU oracle (oracle/) on the seeded config-0 input.
Run:  python tests/golden/make_golden.py      (regression fixture; the paper prints no value for this path)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as orc  # noqa: E402
from paper_2407_16586_b200 import workload as wl  # noqa: E402

if __name__ == "__main__":
    s = wl.make_system(0)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(0))
    pairs, wJ, wK = wl.default_call(D, P, T)
    g, st = orc.gradient(s, pairs, wJ, wK, wl.C_J, wl.C_K, wl.C_LR, wl.OMEGA)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_gradient.txt")
    with open(out, "w") as f:
        f.write("# config 0 (one water, 25 bf) gradient in E_h/bohr, written by tests/golden/make_golden.py from oracle/ only\n")
        f.write("# pairs (D,D),(D,P),(T,T), wJ=2, wK=1, cJ=1, cK=0.157706, cLR=0.842294, omega=0.3; quartets=%d\n" % st["quartets_computed"])
        for row in g:
            f.write(" ".join("%.17e" % v for v in row) + "\n")
    print(open(out).read())
