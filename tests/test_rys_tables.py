"""Host-side check of the generated Rys tables (paper_2407_16586_b200/csrc/rys_meta.inc, rys_tables.inc).

Pin (independent of the generator's Golub-Welsch arithmetic): an n-point Gauss rule for the weight
exp(-T x)/(2 sqrt x) on [0,1] must reproduce the moments F_k(T), k = 0..2n-1 (Rys
quadrature; Boys function = regularised incomplete gamma, scipy).  Evaluated here in double exactly the
way the kernels do (Horner in u = 2 (T - centre)/H; large-T limit beyond TMAX).
"""
import os
import re

import numpy as np
import pytest
from scipy import special

CSRC = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2407_16586_b200", "csrc")


def _load():
    meta = open(os.path.join(CSRC, "rys_meta.inc")).read()
    txt = open(os.path.join(CSRC, "rys_tables.inc")).read()
    deg = int(re.search(r"#define RYS_DEG (\d+)", meta).group(1))
    h = float(re.search(r"#define RYS_H (\S+)", meta).group(1))
    nmax = int(re.search(r"#define RYS_NMAX (\d+)", meta).group(1))
    num = r"[-+]?\d+\.?\d*(?:[eE][-+]?\d+)?"
    tmax = np.array([int(x) for x in re.findall(r"\d+", re.search(r"rys_tmax.*?=\s*\{(.*?)\}", meta).group(1))])
    off = np.array([int(x) for x in re.findall(r"\d+", re.search(r"rys_off.*?=\s*\{(.*?)\}", meta).group(1))])
    body = meta[meta.index("rys_inf(int n, int r)"):]
    inf = [np.array([float(x) for x in re.findall(num, row)]) for row in re.findall(r"\{([^{}]*)\},", body)]
    tab = np.array([float(x) for x in re.findall(num, txt[txt.index("= {"):])])
    return deg, h, nmax, tmax, off, inf, tab


def rys_eval(tables, n, T):
    deg, h, nmax, tmax, off, inf, tab = tables
    if T >= tmax[n]:
        row = inf[n]
        return row[:n] / T, row[n:] / np.sqrt(T)
    i = int(T / h)
    u = (T - (i + 0.5) * h) * (2.0 / h)
    base = off[n] + i * (deg + 1) * 2 * n
    c = tab[base: base + (deg + 1) * 2 * n].reshape(deg + 1, 2 * n)
    v = c[0].copy()
    for k in range(1, deg + 1):
        v = v * u + c[k]
    return v[:n], v[n:]


def boys(k, T):
    if T < 1e-13:
        return 1.0 / (2 * k + 1)
    return special.gammainc(k + 0.5, T) * special.gamma(k + 0.5) / (2.0 * T ** (k + 0.5))


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7])
def test_moments_reproduced(n):
    tables = _load()
    rng = np.random.default_rng(100 + n)
    tmax = tables[3][n]
    Ts = np.concatenate([[0.0, 1e-9, 0.5, 0.999999, 1.0, tmax - 1e-9, tmax, tmax + 3.0, 500.0, 1e5],
                         rng.uniform(0, tmax, 300), rng.uniform(tmax, 3 * tmax, 20)])
    worst = 0.0
    for T in Ts:
        x, w = rys_eval(tables, n, T)
        assert np.all(x > 0) and np.all(x < 1) and np.all(w > 0) and np.all(np.diff(x) > 0)
        for k in range(2 * n):
            ref = boys(k, T)
            err = abs(np.sum(w * x ** k) - ref) / ref
            worst = max(worst, err)
    assert worst < 2e-13, worst
