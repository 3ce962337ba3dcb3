"""Small shared test inputs (no method arithmetic)."""
import numpy as np

from paper_2407_16586_b200 import workload as wl


def tiny_system(with_f=False, tau=0.0):
    xyz = np.array([[0.0, 0.0, 0.0], [1.3, 0.2, -0.4], [-0.5, 1.6, 0.7]])
    a0 = [(0, [3.1, 0.7], [0.4, 0.7]), (1, [0.9], [1.0]), (2, [1.1], [1.0])]
    a1 = [(0, [0.5], [1.0]), (1, [1.7, 0.4], [0.3, 0.8])]
    a2 = [(0, [1.9, 0.3], [0.6, 0.5])]
    if with_f:
        a2.append((3, [0.8], [1.0]))
    return wl.make_custom_system(xyz, [a0, a1, a2], tau=tau)


def two_centre_spdf_system(tau=0.0):
    """Two atoms, each with s, p, d and f shells (two with 2 primitives): every one of the 55 quartet classes occurs,
    (ff|ff) included with shells on different centres."""
    xyz = np.array([[0.0, 0.0, 0.0], [1.1, -0.7, 0.9]])
    a0 = [(0, [2.3, 0.6], [0.5, 0.6]), (1, [1.1], [1.0]), (2, [0.9], [1.0]), (3, [1.3, 0.5], [0.4, 0.7])]
    a1 = [(0, [0.7], [1.0]), (1, [1.9, 0.5], [0.3, 0.8]), (2, [1.4], [1.0]), (3, [0.8], [1.0])]
    return wl.make_custom_system(xyz, [a0, a1], tau=tau)


def densities(nbf, seed=7, n_occ=None):
    return wl.make_densities(nbf, np.random.SeedSequence(seed), n_occ=n_occ)


CALL = dict(cJ=wl.C_J, cK=wl.C_K, cLR=wl.C_LR, omega=wl.OMEGA)
