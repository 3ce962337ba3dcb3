"""GPU parity of the one-electron gradient terms (tdg_onee_gradient; NEXT-4, eq 7 terms 1-3) against the oracle's
orc_onee_gradient, element by element, through the C ABI."""
import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl
from tests.helpers import tiny_system, two_centre_spdf_system

pytestmark = pytest.mark.gpu
TOL_ABS, TOL_REL = 1e-9, 1e-10


@pytest.fixture(scope="module")
def ctx():
    from paper_2407_16586_b200 import tdgrad

    c = tdgrad.Context(0)
    yield c
    c.close()


def _mats(n, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n, n)), rng.standard_normal((n, n))     # general (nonsymmetric) P and W


def _charges(sysm):
    """Nuclear charges of the synthetic systems: the heavier-basis atom of every water is O (8), the others H (1)."""
    nsh = np.bincount(sysm.shells[:, 0], minlength=sysm.natom)
    return np.where(nsh > 3, 8.0, 1.0)


def _check(g, ref):
    scale = max(1.0, float(np.max(np.abs(ref))))
    assert np.max(np.abs(g - ref)) <= max(TOL_ABS, TOL_REL * scale), (np.max(np.abs(g - ref)), scale)


@pytest.mark.parametrize("with_f", [False, True])
def test_tiny_system_all_terms(ctx, orc, with_f):
    s = tiny_system(with_f=with_f)
    Z = np.array([8.0, 1.0, 1.5])
    P, W = _mats(s.nbf, 11)
    ctx.set_system(s)
    ctx.plan(0.0)
    g, _ = ctx.onee_gradient(Z, P, W)
    _check(g, orc.onee_gradient(s, Z, P, W))
    assert np.max(np.abs(g.sum(axis=0))) < 1e-9 * max(1.0, np.max(np.abs(g)))


def test_two_centre_spdf_every_pair_class_and_each_term(ctx, orc):
    s = two_centre_spdf_system()
    Z = np.array([3.0, 2.0])
    P, W = _mats(s.nbf, 5)
    zero = np.zeros_like(P)
    ctx.set_system(s)
    ctx.plan(0.0)
    for Zv, Pv, Wv in ((Z, P, W), (np.zeros(2), zero, W), (np.zeros(2), P, zero), (Z, P, zero), (Z, zero, zero)):
        g, _ = ctx.onee_gradient(Zv, Pv, Wv)
        _check(g, orc.onee_gradient(s, Zv, Pv, Wv))
    g_none, _ = ctx.onee_gradient(Z, None, None)          # nuclear repulsion alone
    _check(g_none, orc.onee_gradient(s, Z, zero, zero))


def test_cfg0_and_cfg1_water_clusters(ctx, orc):
    import torch

    for cfg in (0, 1):
        s = wl.make_system(cfg)
        Z = _charges(s)
        P, W = _mats(s.nbf, 20 + cfg)
        ctx.set_system(s)
        ctx.plan(0.0)
        ref = orc.onee_gradient(s, Z, P, W)
        g, _ = ctx.onee_gradient(Z, P, W)
        _check(g, ref)
        # device-resident inputs and output
        out = torch.zeros((s.natom, 3), dtype=torch.float64, device="cuda")
        g2, ms = ctx.onee_gradient(Z, torch.from_numpy(P).cuda(), torch.from_numpy(W).cuda(), out=out)
        _check(g2.cpu().numpy(), ref)
        assert ms > 0.0
    # the plan's own screening (tau = 1e-14 at cfg 1) drops only pairs whose one-electron integrals are negligible
    ctx.plan(s.tau, s.density_weighted)
    g3, _ = ctx.onee_gradient(Z, P, W)
    _check(g3, ref)


def test_spherical_shells(ctx, orc):
    """Flagged d/f shells: P and W are given in the mixed spherical basis; the library back-transforms them (NEXT-2)."""
    s = two_centre_spdf_system()
    flags = np.array([1 if l >= 2 else 0 for l in s.shells[:, 1]], dtype=np.int32)
    Cm = orc.sph_transform(s, flags)                       # [nbf_in, nbf_cart]
    nin = Cm.shape[0]
    P, W = _mats(nin, 9)
    Z = np.array([2.0, 1.0])
    ctx.set_system(s)
    ctx.set_spherical(flags)
    ctx.plan(0.0)
    g, _ = ctx.onee_gradient(Z, P, W)
    ctx.set_spherical(None)
    _check(g, orc.onee_gradient(s, Z, Cm.T @ P @ Cm, Cm.T @ W @ Cm))


def test_many_atoms_spans_several_nucleus_chunks(ctx, orc):
    """More than 256 nuclei (the kernel's chunk) with a ragged tail: 96 waters = 288 atoms, s/p shells only to keep the oracle fast."""
    rng = np.random.default_rng(3)
    xyz = wl.water_cluster_xyz(96, rng)
    shells = []
    for a in range(xyz.shape[0]):
        shells.append([(0, [1.1, 0.3], [0.5, 0.6]), (1, [0.7], [1.0])] if a % 3 == 0 else [(0, [0.6], [1.0])])
    s = wl.make_custom_system(xyz, shells)
    Z = np.where(np.arange(s.natom) % 3 == 0, 8.0, 1.0)
    P, W = _mats(s.nbf, 13)
    ctx.set_system(s)
    ctx.plan(1e-13)
    g, _ = ctx.onee_gradient(Z, P, W)
    _check(g, orc.onee_gradient(s, Z, P, W))
