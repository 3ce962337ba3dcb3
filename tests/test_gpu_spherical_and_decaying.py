"""GPU parity for the two other "next" rows of SURVEY.md 8(f):
NEXT-2 spherical-harmonic shells (tdg_set_spherical: density back-transform D_cart = C^T D_sph C inside the library; the oracle
side back-transforms in numpy with its own solid-harmonic table and runs Cartesian) and NEXT-4 spatially decaying densities
(workload.make_decaying_densities), where the density-weighted test actually prunes."""
import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl
from tests.helpers import CALL, tiny_system, two_centre_spdf_system

pytestmark = pytest.mark.gpu
ABS_TOL, REL_TOL = 1e-9, 1e-10


@pytest.fixture(scope="module")
def ctx():
    from paper_2407_16586_b200 import tdgrad

    c = tdgrad.Context(0)
    yield c
    c.close()


def _compare(g, ref):
    d = np.max(np.abs(g - ref))
    assert d <= ABS_TOL, d
    assert d / np.max(np.abs(ref)) <= REL_TOL, d / np.max(np.abs(ref))


@pytest.mark.parametrize("system,flags", [("tiny_f", "all"), ("two_centre", "all"), ("two_centre", "mixed")])
def test_spherical_gradient_and_energy(ctx, orc, system, flags):
    s = tiny_system(with_f=True) if system == "tiny_f" else two_centre_spdf_system()
    fl = np.ones(s.nshell, dtype=np.int32)
    if flags == "mixed":
        fl[::2] = 0
    C = orc.sph_transform(s, fl)
    nin = C.shape[0]
    rng = np.random.default_rng(3)
    M = [rng.standard_normal((nin, nin)) for _ in range(3)]
    pairs = [(M[0] + M[0].T, M[1]), (M[2], M[2])]
    wJ, wK = np.array([2.0, 0.7]), np.array([1.0, -1.4])
    ctx.set_system(s)
    ctx.set_spherical(fl)
    assert ctx.nbf() == nin
    ctx.plan(0.0, 0)
    g, st = ctx.gradient(pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    e = ctx.energy(pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    cart = [(C.T @ a @ C, C.T @ b @ C) for a, b in pairs]
    ref, _ = orc.gradient(s, cart, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    eref, _ = orc.energy(s, cart, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    _compare(g, ref)
    assert abs(e - eref) <= 1e-11 * max(1.0, abs(eref))
    ctx.set_spherical(None)
    assert ctx.nbf() == s.nbf


def test_spherical_fock(ctx, orc):
    s = two_centre_spdf_system()
    fl = np.ones(s.nshell, dtype=np.int32)
    C = orc.sph_transform(s, fl)
    nin = C.shape[0]
    rng = np.random.default_rng(4)
    B = [rng.standard_normal((nin, nin)) for _ in range(2)]
    w = (np.array([4.0, 2.0]), np.array([1.0, 1.0]), np.array([1.0, 0.0]))
    ctx.set_system(s)
    ctx.set_spherical(fl)
    ctx.plan(0.0, 0)
    F, st = ctx.fock(B, *w, wl.C_K, wl.C_LR, wl.OMEGA)
    R, _ = orc.fock(s, [C.T @ b @ C for b in B], *w, wl.C_K, wl.C_LR, wl.OMEGA, tau=0.0)
    for f, r in zip(F, R):
        rs = C @ r @ C.T
        assert f.shape == (nin, nin)
        assert np.abs(f - rs).max() <= 1e-10 * np.abs(rs).max()
    ctx.set_spherical(None)


def test_cfg2_geometry_spherical_subsample(ctx, orc):
    """32 waters with f shells, every d and f shell spherical (the paper's production basis is spherical)."""
    s = wl.make_system(2)
    fl = np.ones(s.nshell, dtype=np.int32)
    C = orc.sph_transform(s, fl)
    nin = C.shape[0]
    D, P, T = wl.make_densities(nin, wl.density_seed(2))
    pairs, wJ, wK = wl.default_call(D, P, T)
    ctx.set_system(s)
    ctx.set_spherical(fl)
    ctx.plan(s.tau, s.density_weighted, 3000, 5)
    g, st = ctx.gradient(pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    cart = [(C.T @ a @ C, C.T @ b @ C) for a, b in pairs]
    ref, rst = orc.gradient(s, cart, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"], sample_mod=3000, sample_seed=5)
    _compare(g, ref)
    assert st["quartets_computed"] == rst["quartets_computed"]
    ctx.set_spherical(None)


@pytest.mark.parametrize("tau", [1e-9, 1e-7])
def test_decaying_densities_cfg1_density_weighted(ctx, orc, tau):
    """NEXT-4: with spatially decaying densities the density-weighted test (S9) removes most Schwarz survivors; both sides must
    drop the same quartets (counts within a handful of edge flips) and agree on the gradient."""
    s = wl.make_system(1)
    D, P, T = wl.make_decaying_densities(s, 11)
    pairs, wJ, wK = wl.default_call(D, P, T)
    ctx.set_system(s)
    ctx.plan(tau, 1)
    g, st = ctx.gradient(pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    ref, rst = orc.gradient(s, pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"], tau=tau, density_weighted=1)
    _compare(g, ref)
    assert st["quartets_visited"] == rst["quartets_visited"]
    assert abs(st["quartets_computed"] - rst["quartets_computed"]) <= 5
    assert st["quartets_computed"] < 0.8 * st["quartets_visited"]          # the weight prunes


@pytest.mark.slow
def test_decaying_densities_cfg3_subsample(ctx, orc):
    s = wl.make_system(3)
    D, P, T = wl.make_decaying_densities(s, 13)
    pairs, wJ, wK = wl.default_call(D, P, T)
    ctx.set_system(s)
    ctx.plan(s.tau, s.density_weighted, 20000, 9)
    g, st = ctx.gradient(pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    ref, rst = orc.gradient(s, pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"], sample_mod=20000, sample_seed=9)
    _compare(g, ref)
    assert st["pairs_kept"] == rst["pairs_kept"]
    assert abs(st["quartets_computed"] - rst["quartets_computed"]) <= 3
