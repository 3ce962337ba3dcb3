"""Pins for the oracle's Fock-type build (NEXT-1; eq 19, eqs 33-34).

  F[mn] = sum_ls [ wJ B[sl] (mn|ls) - (wK B + wKT B^T)[sl] ( cK (ml|sn) + cLR (ml|sn)_lr ) ]

Pinned by: numpy einsum over orc_eri_tensor (the definition, written with a library contraction); the contracted energy
sum_mn A[mn] F[B][mn] = J/K combination of orc_energy (an oracle function with its own pins); symmetry of F for symmetric B;
the MO-basis sigma vector of eq 33 built from eq 17's (ia|jb), (ij|ab), (ib|aj) integrals; the unique-quartet loop with its
8-fold digestion against the plain nshell^4 loop; screening limits."""
import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl
from tests.helpers import tiny_system, two_centre_spdf_system

OMEGA = 0.3


def _mats(n, seed, k=2):
    rng = np.random.default_rng(seed)
    return [rng.standard_normal((n, n)) for _ in range(k)]


@pytest.mark.parametrize("with_f", [False, True])
def test_fock_vs_einsum_over_eri_tensor(orc, with_f):
    s = tiny_system(with_f=with_f)
    n = s.nbf
    B = _mats(n, 1, 2)
    wJ, wK, wKT, cK, cLR = np.array([4.0, 2.0]), np.array([1.0, 1.0]), np.array([1.0, 0.0]), 0.3, 0.6
    g, glr = orc.eri_tensor(s), orc.eri_tensor(s, omega=OMEGA)
    gk = cK * g + cLR * glr
    F, st = orc.fock(s, B, wJ, wK, wKT, cK, cLR, OMEGA)
    F4 = orc.fock_n4(s, B, wJ, wK, wKT, cK, cLR, OMEGA)
    for m in range(2):
        X = wK[m] * B[m] + wKT[m] * B[m].T
        ref = wJ[m] * np.einsum("sl,mnls->mn", B[m], g) - np.einsum("sl,mlsn->mn", X, gk)
        scale = np.abs(ref).max()
        assert np.abs(F4[m] - ref).max() <= 1e-12 * scale
        assert np.abs(F[m] - ref).max() <= 1e-12 * scale
    # eq 34's second exchange pattern (ms|ln) with B is the first pattern with B^T
    ref34 = np.einsum("sl,mlsn->mn", B[0], g) + np.einsum("sl,msln->mn", B[0], g)
    got = orc.fock_n4(s, [B[0]], np.zeros(1), np.ones(1), np.ones(1), 1.0, 0.0, OMEGA)[0]
    assert np.abs(-got - ref34).max() <= 1e-12 * np.abs(ref34).max()


def test_fock_contracted_with_a_density_is_the_energy(orc):
    """sum_mn A[mn] F[B][mn] with (wJ, wK, wKT) = (1, 1, 0) equals J(A,B') - cK K - cLR K_lr of orc_energy for the index
    pattern of the energy: J(A,B) = sum A_mn B_ls (mn|ls), K(A,B) = sum A_ml B_ns (mn|ls)."""
    s = tiny_system(with_f=True)
    n = s.nbf
    A, B = _mats(n, 2, 2)
    cK, cLR = 0.25, 0.7
    F = orc.fock_n4(s, [B], np.ones(1), np.ones(1), np.zeros(1), cK, cLR, OMEGA)[0]
    lhs = float(np.sum(A * F))
    # sum_mn A_mn sum_ls B_sl (mn|ls) = J(A, B^T);  sum_mn A_mn sum_ls B_sl (ml|sn) = sum A_mn B_sl (ml|sn): relabel (ml|sn)->(mn|ls)
    # with n<->l: sum A_ml B_sn ... = K(A, B^T) in the energy's convention K(A,B) = sum A_ml B_ns (mn|ls)
    e, _ = orc.energy(s, [(A, B.T.copy())], np.ones(1), np.ones(1), 1.0, cK, cLR, OMEGA)
    assert lhs == pytest.approx(e, rel=1e-12)


def test_fock_symmetry(orc):
    s = two_centre_spdf_system()
    n = s.nbf
    B = _mats(n, 3, 1)[0]
    Bs = B + B.T
    F, _ = orc.fock(s, [Bs, B], np.array([2.0, 2.0]), np.array([1.0, 1.0]), np.array([0.0, 1.0]), 0.2, 0.8, OMEGA)
    assert np.abs(F[0] - F[0].T).max() <= 1e-13 * np.abs(F[0]).max()     # symmetric B: symmetric F
    assert np.abs(F[1] - F[1].T).max() <= 1e-13 * np.abs(F[1]).max()     # wK = wKT: K[B] + K[B^T] is symmetric too
    Fn, _ = orc.fock(s, [B], np.array([0.0]), np.array([1.0]), np.array([0.0]), 1.0, 0.0, OMEGA)
    assert np.abs(Fn[0] - Fn[0].T).max() > 1e-3 * np.abs(Fn[0]).max()   # a nonsymmetric B alone gives a nonsymmetric K
    F4 = orc.fock_n4(s, [Bs, B], np.array([2.0, 2.0]), np.array([1.0, 1.0]), np.array([0.0, 1.0]), 0.2, 0.8, OMEGA)
    for a, b in zip(F, F4):
        assert np.abs(a - b).max() <= 1e-12 * np.abs(b).max()


def test_sigma_vector_of_eq_33_in_the_mo_basis(orc):
    """sigma = A b with A_ai,bj = 4(ia|jb) - alpha[(ij|ab) + (ib|aj)] - beta[...]_lr (eq 17 without d and f_XC) equals
    C_v^T F~[B] C_o with B = C_v b C_o^T (eqs 33-34)."""
    s = tiny_system()
    n = s.nbf
    rng = np.random.default_rng(4)
    q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    no = 5
    Co, Cv = q[:, :no], q[:, no:]
    b = rng.standard_normal((n - no, no))
    alpha, beta = 0.157706, 0.842294
    g, glr = orc.eri_tensor(s), orc.eri_tensor(s, omega=OMEGA)
    sig = np.zeros_like(b)
    for gg, coef in ((g, alpha), (glr, beta)):
        ijab = np.einsum("mi,nj,la,sb,mnls->ijab", Co, Co, Cv, Cv, gg, optimize=True)
        ibaj = np.einsum("mi,nb,la,sj,mnls->ibaj", Co, Cv, Cv, Co, gg, optimize=True)
        sig -= coef * (np.einsum("ijab,bj->ai", ijab, b) + np.einsum("ibaj,bj->ai", ibaj, b))
    iajb = np.einsum("mi,na,lj,sb,mnls->iajb", Co, Cv, Co, Cv, g, optimize=True)
    sig += 4.0 * np.einsum("iajb,bj->ai", iajb, b)
    B = Cv @ b @ Co.T
    F = orc.fock_n4(s, [B], np.array([4.0]), np.ones(1), np.ones(1), alpha, beta, OMEGA)[0]
    got = Cv.T @ F @ Co
    assert np.abs(got - sig).max() <= 1e-11 * np.abs(sig).max()


def test_fock_screening_limits(orc):
    s0 = wl.make_system(1)
    keep = s0.shells[:, 0] < 6
    s = wl.System(s0.xyz[:6], s0.shells[keep], s0.exps, s0.coefs)
    B = _mats(s.nbf, 6, 1)
    w = (np.array([4.0]), np.ones(1), np.ones(1), wl.C_K, wl.C_LR, wl.OMEGA)
    F0, st0 = orc.fock(s, B, *w, tau=0.0)
    F1, st1 = orc.fock(s, B, *w, tau=1e-30)
    assert np.abs(F0[0] - F1[0]).max() <= 1e-12 * np.abs(F0[0]).max()
    F2, st2 = orc.fock(s, B, *w, tau=1e-7)
    F3, st3 = orc.fock(s, B, *w, tau=1e-7, density_weighted=1)
    assert st2["quartets_computed"] < st0["quartets_computed"]
    assert st3["quartets_computed"] <= st2["quartets_computed"] and st3["quartets_visited"] == st2["quartets_visited"]
    dropped = st0["quartets_computed"] - st3["quartets_computed"]
    assert np.abs(F3[0] - F0[0]).max() <= 1e-7 * 36 * 8 * max(1, dropped) ** 0.5 * 10   # each dropped integral x density < tau
    # subsample partitions: the m residue classes of the hash add up to the full matrix
    parts = [orc.fock(s, B, *w, tau=1e-7, sample_mod=3, sample_seed=sd)[0][0] for sd in (1,)]
    assert np.abs(parts[0]).max() < np.abs(F2[0]).max() * 1.01
