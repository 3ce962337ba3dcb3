"""Pins for the oracle's contraction and gradient (O8-O10): finite differences of the contracted energy
(the paper's own validation), translational invariance, the N^4 loop vs the
unique-quartet loop, Gamma index conventions (eqs 2-5, 106 eq 12, 110-114 eqs 13-14)."""
import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl
from tests.helpers import CALL, densities, tiny_system


def _args(D, P, T):
    pairs, wJ, wK = wl.default_call(D, P, T)
    return pairs, wJ, wK


def test_energy_vs_einsum_over_eri_tensor(orc):
    """orc_energy against the plain definition (E) evaluated with numpy on the full tensor."""
    s = tiny_system(with_f=True)
    D, P, T = densities(s.nbf)
    pairs, wJ, wK = _args(D, P, T)
    g, glr = orc.eri_tensor(s), orc.eri_tensor(s, omega=CALL["omega"])
    ref = 0.0
    for (A, B), wj, wk in zip(pairs, wJ, wK):
        J = np.einsum("mn,ls,mnls->", A, B, g)
        K = np.einsum("ml,ns,mnls->", A, B, g)
        Klr = np.einsum("ml,ns,mnls->", A, B, glr)
        ref += wj * CALL["cJ"] * J - wk * (CALL["cK"] * K + CALL["cLR"] * Klr)
    e, st = orc.energy(s, pairs, wJ, wK, **CALL)
    assert e == pytest.approx(ref, rel=1e-12)
    assert st["quartets_computed"] == (lambda n: n * (n + 1) // 2)(s.nshell * (s.nshell + 1) // 2)


def test_exchange_index_convention_mo_sum(orc):
    """K(T,T) = sum_{ia,jb} X_ia X_jb (ij|ab) and J(T,T) = sum X_ia X_jb (ia|jb) with T = C_o X C_v^T (reading S2)."""
    s = tiny_system()
    n = s.nbf
    rng = np.random.default_rng(3)
    q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    no = 4
    Co, Cv = q[:, :no], q[:, no:]
    X = rng.standard_normal((no, n - no))
    T = Co @ X @ Cv.T
    g = orc.eri_tensor(s)
    ijab = np.einsum("mi,nj,la,sb,mnls->ijab", Co, Co, Cv, Cv, g, optimize=True)
    iajb = np.einsum("mi,na,lj,sb,mnls->iajb", Co, Cv, Co, Cv, g, optimize=True)
    K_mo = np.einsum("ia,jb,ijab->", X, X, ijab)
    J_mo = np.einsum("ia,jb,iajb->", X, X, iajb)
    one, zero = np.ones(1), np.zeros(1)
    eK, _ = orc.energy(s, [(T, T)], zero, one, 1.0, 1.0, 0.0, 0.3)   # E = -K
    eJ, _ = orc.energy(s, [(T, T)], one, zero, 1.0, 1.0, 0.0, 0.3)   # E = +J
    assert -eK == pytest.approx(K_mo, rel=1e-12)
    assert eJ == pytest.approx(J_mo, rel=1e-12)
    K_other = np.einsum("ms,ln,mnls->", T, T, g)  # the (ib|ja)-type pattern TDA drops: must differ
    assert abs(K_other - K_mo) > 1e-3 * abs(K_mo)


@pytest.mark.parametrize("with_f", [False, True])
def test_gradient_vs_finite_difference_of_energy(orc, with_f):
    s = tiny_system(with_f=with_f)
    D, P, T = densities(s.nbf)
    pairs, wJ, wK = _args(D, P, T)
    g, _ = orc.gradient(s, pairs, wJ, wK, **CALL)
    h = 1e-4
    fd = np.zeros_like(g)
    for a in range(s.natom):
        for x in range(3):
            ep = em = 0.0
            for sign in (+1, -1):
                xyz = s.xyz.copy()
                xyz[a, x] += sign * h
                e, _ = orc.energy(wl.System(xyz, s.shells, s.exps, s.coefs), pairs, wJ, wK, **CALL)
                if sign > 0:
                    ep = e
                else:
                    em = e
            fd[a, x] = (ep - em) / (2 * h)
    assert np.abs(fd - g).max() <= 1e-6
    assert np.abs(g.sum(axis=0)).max() <= 1e-10


def test_n4_loop_equals_unique_quartet_loop(orc):
    """'8-fold permutational symmetry on tiny inputs' (BASELINE.json): plain nshell^4 loop with the plain Gamma
    equals the unique-quartet loop with the symmetrised Gamma-tilde and degeneracy weights."""
    for s in (wl.make_system(0), tiny_system(with_f=True)):
        D, P, T = densities(s.nbf, seed=11)
        pairs, wJ, wK = _args(D, P, T)
        g, _ = orc.gradient(s, pairs, wJ, wK, **CALL)
        g4 = orc.gradient_n4(s, pairs, wJ, wK, **CALL)
        assert np.abs(g - g4).max() <= 2e-13 * max(1.0, np.abs(g).max())
        assert np.abs(g4.sum(axis=0)).max() <= 1e-10


def test_operator_limits_and_linearity(orc):
    s = tiny_system()
    D, P, T = densities(s.nbf, seed=5)
    pairs, wJ, wK = _args(D, P, T)
    # omega = 1e6: the lr gradient equals the full one, so (cK=0,cLR=c) == (cK=c,cLR=0)
    a, _ = orc.gradient(s, pairs, wJ, wK, 1.0, 0.0, 0.7, 1e6)
    b, _ = orc.gradient(s, pairs, wJ, wK, 1.0, 0.7, 0.0, 0.3)
    assert np.abs(a - b).max() <= 1e-10 * np.abs(b).max()
    # linearity in (wJ, wK) and in the pair list
    g1, _ = orc.gradient(s, pairs[:1], wJ[:1], wK[:1], **CALL)
    g2, _ = orc.gradient(s, pairs[1:], wJ[1:], wK[1:], **CALL)
    g12, _ = orc.gradient(s, pairs, wJ, wK, **CALL)
    assert np.abs(g1 + g2 - g12).max() <= 1e-12 * np.abs(g12).max()
    g3, _ = orc.gradient(s, pairs, 3 * wJ, 3 * wK, **CALL)
    assert np.abs(g3 - 3 * g12).max() <= 1e-12 * np.abs(g12).max()
    # J is insensitive to transposes, K(T,T) is not (reading S2)
    one, zero = np.ones(1), np.zeros(1)
    gj, _ = orc.gradient(s, [(T, T)], one, zero, 1.0, 0.0, 0.0, 0.3)
    gjt, _ = orc.gradient(s, [(T.T.copy(), T)], one, zero, 1.0, 0.0, 0.0, 0.3)
    assert np.abs(gj - gjt).max() <= 1e-13 * np.abs(gj).max()


def test_screening_limits_and_counts(orc):
    s = wl.make_system(1)
    keep = s.shells[:, 0] < 6  # two waters of config 1
    s = wl.System(s.xyz[:6], s.shells[keep], s.exps, s.coefs)
    D, P, T = densities(s.nbf, seed=9)
    pairs, wJ, wK = _args(D, P, T)
    g0, st0 = orc.gradient(s, pairs, wJ, wK, **CALL, tau=0.0)
    g1, st1 = orc.gradient(s, pairs, wJ, wK, **CALL, tau=1e-30)
    assert np.abs(g0 - g1).max() <= 1e-12 * np.abs(g0).max()
    g2, st2 = orc.gradient(s, pairs, wJ, wK, **CALL, tau=1e-6)
    assert st2["quartets_computed"] < st0["quartets_computed"]
    assert np.abs(g0 - g2).max() < 1e-2  # screened result stays close (error ~ tau x dropped)
    g3, st3 = orc.gradient(s, pairs, wJ, wK, **CALL, tau=1e-6, density_weighted=1)
    assert st3["quartets_computed"] <= st2["quartets_computed"]
    assert st3["quartets_visited"] == st2["quartets_visited"]
    # Schwarz bound is a bound: |(mn|ls)| <= Q_mn Q_ls on a sample of shell quartets
    Q = orc.schwarz(s)
    rng = np.random.default_rng(0)
    for _ in range(40):
        i, j, k, l = rng.integers(0, s.nshell, 4)
        v = np.abs(orc.eri_shell(s, i, j, k, l)).max()
        assert v <= Q[i, j] * Q[k, l] * (1 + 1e-12)


def test_subsample_rule(orc):
    """S12: deterministic keep rule, symmetric in the canonical indices, about 1/m of quartets."""
    m, seed = 7, 12345
    n = 14
    cnt = tot = 0
    for i in range(n):
        for j in range(i + 1):
            for k in range(n):
                for l in range(k + 1):
                    a = orc.sample_keep(i, j, k, l, m, seed)
                    assert a == orc.sample_keep(j, i, l, k, m, seed) == orc.sample_keep(k, l, i, j, m, seed)
                    cnt += a
                    tot += 1
    assert abs(cnt / tot - 1 / m) < 0.02
    s = tiny_system()
    D, P, T = densities(s.nbf)
    pairs, wJ, wK = _args(D, P, T)
    total = np.zeros((s.natom, 3))
    # the m residue classes partition the quartets: summing over seeds is not a partition, so check counts only
    g, st = orc.gradient(s, pairs, wJ, wK, **CALL, sample_mod=m, sample_seed=seed)
    gall, stall = orc.gradient(s, pairs, wJ, wK, **CALL)
    assert 0 < st["quartets_computed"] < stall["quartets_computed"]
