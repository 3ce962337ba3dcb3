"""Pins for the oracle's density-weighted screening rule (reading S9 of DESIGN.md):
shell-block maxima d_ij (`density_maxima`) and W_ijkl = max(C_J d_ij d_kl, C_K max(d_ik d_jl, d_il d_jk)).

What fixes them, independently of the oracle's own arithmetic:
  * the mathematics: Q_ij Q_kl W_ijkl must bound every J-type and every K-type density-weighted integral of the
    shell quartet (Cauchy-Schwarz on the integral, block maxima on the densities) -- with nonsymmetric matrices of
    widely varying block magnitudes a weight taken on the wrong shells, on one orientation only, or with |cLR| or a
    pair weight missing, violates it;
  * a closed-form special case: with s shells only, one symmetric matrix and one of the two terms switched off, the
    bound is attained exactly (W = |w c| |A_ij| |A_kl|  resp.  (|cK|+|cLR|)|w| max(|A_ik A_jl|, |A_il A_jk|));
  * invariance: the 8 index permutations of a quartet and transposing every matrix leave W unchanged;
  * the error it causes: |g(tau, weighted) - g(unscreened)| <= c * n_dropped * tau with the constant stated below.
"""
import itertools

import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl
from tests.helpers import tiny_system


def _shell_slices(s):
    off = np.concatenate([[0], np.cumsum([(l + 1) * (l + 2) // 2 for l in s.shells[:, 1]])])
    return [slice(int(off[i]), int(off[i + 1])) for i in range(s.nshell)]


def _ragged_matrices(nbf, seed, nmat):
    """Nonsymmetric matrices whose rows/columns span four orders of magnitude (so block maxima differ a lot)."""
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(nmat):
        r = 10.0 ** rng.uniform(-2, 0, nbf)
        c = 10.0 ** rng.uniform(-2, 0, nbf)
        out.append(np.ascontiguousarray(r[:, None] * rng.standard_normal((nbf, nbf)) * c[None, :]))
    return out


@pytest.mark.parametrize("cK,cLR", [(0.3, 0.6), (0.0, 0.8), (0.7, 0.0)])
def test_weighted_bound_dominates_every_density_weighted_integral(orc, cK, cLR):
    """For EVERY ordered shell quartet of a 3-atom s/p/d/f system and every function quartet in it:
         |sum_k wJ_k cJ A_mn B_ls (mn|ls)|                              <= Q_ij Q_kl C_J d_ij d_kl   <= Q Q W
         |sum_k wK_k A_ml B_ns (cK (mn|ls) + cLR (mn|ls)_lr)|           <= Q_ij Q_kl C_K d_ik d_jl   <= Q Q W
         |sum_k wK_k A_ms B_nl (cK (mn|ls) + cLR (mn|ls)_lr)|           <= Q_ij Q_kl C_K d_il d_jk   <= Q Q W
       with the integrals from orc_eri_tensor, the density products from the n^4 definition in numpy."""
    s = tiny_system(with_f=True)
    n, ns = s.nbf, s.nshell
    A1, B1, A2, B2 = _ragged_matrices(n, 5, 4)
    pairs = [(A1, B1), (A2, B2)]
    wJ, wK, cJ, omega = np.array([2.0, -0.7]), np.array([1.0, 1.6]), 0.9, 0.3
    d, W = orc.density_weights(s, pairs, wJ, wK, cJ, cK, cLR)
    Q = orc.schwarz(s)
    g, glr = orc.eri_tensor(s), orc.eri_tensor(s, omega=omega)
    gk = cK * g + cLR * glr
    TJ = sum(wj * cJ * np.einsum("mn,ls->mnls", A, B) for (A, B), wj in zip(pairs, wJ)) * g
    TK1 = sum(wk * np.einsum("ml,ns->mnls", A, B) for (A, B), wk in zip(pairs, wK)) * gk
    TK2 = sum(wk * np.einsum("ms,nl->mnls", A, B) for (A, B), wk in zip(pairs, wK)) * gk
    sl = _shell_slices(s)
    tight = 0.0
    for i, j, k, l in itertools.product(range(ns), repeat=4):
        blk = (sl[i], sl[j], sl[k], sl[l])
        bound = Q[i, j] * Q[k, l] * W[i, j, k, l] * (1 + 1e-12) + 1e-300
        for X in (TJ, TK1, TK2):
            v = np.abs(X[blk]).max()
            assert v <= bound, (i, j, k, l)
            tight = max(tight, v / bound)
    assert tight > 0.05       # the bound is not vacuous (a weight inflated to the global maximum would be)


def test_block_maxima_cover_both_orientations_and_all_matrices(orc):
    """d_ij against the definition written with numpy slices: max over A_k, B_k, both (i,j) and (j,i) blocks."""
    s = tiny_system(with_f=True)
    mats = _ragged_matrices(s.nbf, 11, 4)
    pairs = [(mats[0], mats[1]), (mats[2], mats[3])]
    d, _ = orc.density_weights(s, pairs, np.ones(2), np.ones(2), 1.0, 1.0, 1.0, want_W=False)
    sl = _shell_slices(s)
    assert np.array_equal(d, d.T)
    for i in range(s.nshell):
        for j in range(s.nshell):
            ref = max(max(np.abs(M[sl[i], sl[j]]).max(), np.abs(M[sl[j], sl[i]]).max()) for M in mats)
            assert d[i, j] == ref
    # every matrix matters: blow up one element of each in turn
    for q in range(4):
        mats2 = [m.copy() for m in mats]
        mats2[q][sl[3].start, sl[5].start] = 1e3
        d2, _ = orc.density_weights(s, [(mats2[0], mats2[1]), (mats2[2], mats2[3])], np.ones(2), np.ones(2), 1.0, 1.0, 1.0, want_W=False)
        assert d2[3, 5] == 1e3 and d2[5, 3] == 1e3


def _s_only_system():
    xyz = np.array([[0.0, 0.0, 0.0], [1.4, 0.1, -0.3], [-0.6, 1.5, 0.8], [0.4, -1.1, 1.2]])
    atoms = [[(0, [2.1, 0.6], [0.5, 0.6]), (0, [0.3], [1.0])], [(0, [0.9], [1.0])], [(0, [1.3, 0.4], [0.4, 0.7])], [(0, [0.5], [1.0])]]
    return wl.make_custom_system(xyz, atoms)


def test_weight_closed_form_for_s_shells(orc):
    """s shells only, one symmetric matrix, (A, A): with K off the weight IS |wJ cJ A_ij A_kl|; with J off it IS
    (|cK|+|cLR|) |wK| max(|A_ik A_jl|, |A_il A_jk|) (one function per shell: block maxima are the elements)."""
    s = _s_only_system()
    ns = s.nshell
    rng = np.random.default_rng(2)
    A = rng.standard_normal((ns, ns)); A = A + A.T
    wJ, wK = np.array([1.7]), np.array([0.6])
    _, WJ = orc.density_weights(s, [(A, A)], wJ, np.zeros(1), 0.8, 0.2, 0.5)
    _, WK = orc.density_weights(s, [(A, A)], np.zeros(1), wK, 0.8, 0.2, 0.5)
    _, Wb = orc.density_weights(s, [(A, A)], wJ, wK, 0.8, 0.2, 0.5)
    a = np.abs(A)
    refJ = 1.7 * 0.8 * np.einsum("ij,kl->ijkl", a, a)
    refK = (0.2 + 0.5) * 0.6 * np.maximum(np.einsum("ik,jl->ijkl", a, a), np.einsum("il,jk->ijkl", a, a))
    assert np.allclose(WJ, refJ, rtol=1e-15, atol=0)
    assert np.allclose(WK, refK, rtol=1e-15, atol=0)
    assert np.allclose(Wb, np.maximum(refJ, refK), rtol=1e-15, atol=0)


def test_weight_is_invariant_under_quartet_permutations_and_transposes(orc):
    s = tiny_system()
    mats = _ragged_matrices(s.nbf, 3, 2)
    args = (np.array([2.0]), np.array([1.0]), 1.0, 0.2, 0.8)
    d, W = orc.density_weights(s, [(mats[0], mats[1])], *args)
    dT, WT = orc.density_weights(s, [(mats[0].T.copy(), mats[1].T.copy())], *args)
    dS, WS = orc.density_weights(s, [(mats[1], mats[0])], *args)
    assert np.array_equal(d, dT) and np.array_equal(W, WT)
    assert np.array_equal(d, dS) and np.array_equal(W, WS)
    for perm in ("jikl", "ijlk", "jilk", "klij", "lkij", "klji", "lkji"):
        assert np.array_equal(W, np.einsum("ijkl->" + perm, W)), perm


def test_weighted_screening_error_is_bounded_by_dropped_times_tau(orc):
    """|g(tau, density-weighted) - g(unscreened)|_max <= c * n_dropped * tau.  Each dropped quartet has
    |Gt (mn|ls)| < tau for every function quartet; its gradient contribution replaces the integral by a centre
    derivative, at most ~2 sqrt(2 zeta_max) (l+1) times larger per centre (here zeta_max = 5000: ~300), times the
    number of function quartets and the J + 2 K terms of the symmetrised product -- but the dropped quartets are the
    far-apart diffuse ones, where the derivative is SMALLER than the integral, and their errors do not add coherently:
    the measured ratio (printed with -s) is ~1e-3, and the test states c = 1."""
    s0 = wl.make_system(1)
    keep = s0.shells[:, 0] < 9          # three waters of config 1: 36 shells
    s = wl.System(s0.xyz[:9], s0.shells[keep], s0.exps, s0.coefs)
    D, P, T = wl.make_densities(s.nbf, np.random.SeedSequence(9))
    pairs, wJ, wK = wl.default_call(D, P, T)
    call = dict(cJ=wl.C_J, cK=wl.C_K, cLR=wl.C_LR, omega=wl.OMEGA)
    g0, st0 = orc.gradient(s, pairs, wJ, wK, **call, tau=0.0)
    worst = 0.0
    for tau in (1e-9, 1e-7, 1e-5):
        g1, st1 = orc.gradient(s, pairs, wJ, wK, **call, tau=tau, density_weighted=1)
        dropped = st0["quartets_computed"] - st1["quartets_computed"]
        assert dropped > 0
        err = np.abs(g1 - g0).max()
        assert err <= 1.0 * dropped * tau
        worst = max(worst, err / (dropped * tau))
        # and the weighted rule only ever drops quartets the Schwarz-only rule would keep or drop: never computes more
        g2, st2 = orc.gradient(s, pairs, wJ, wK, **call, tau=tau, density_weighted=0)
        assert st1["quartets_computed"] <= st2["quartets_computed"]
    print("max |dg| / (n_dropped tau) =", worst)


def test_keep_decision_matches_weights(orc):
    """The quartet count of the weighted run equals the count of canonical quartets with Q Q >= tau and Q Q W >= tau,
    W and Q taken from the exported arrays (ties the exported W to the rule contract_driver applies)."""
    s = tiny_system(with_f=True)
    D, P, T = wl.make_densities(s.nbf, np.random.SeedSequence(4))
    pairs, wJ, wK = wl.default_call(D, P, T)
    call = dict(cJ=wl.C_J, cK=wl.C_K, cLR=wl.C_LR, omega=wl.OMEGA)
    Q = orc.schwarz(s)
    _, W = orc.density_weights(s, pairs, wJ, wK, wl.C_J, wl.C_K, wl.C_LR)
    ns = s.nshell
    for tau in (1e-6, 1e-4, 1e-3):
        _, st = orc.gradient(s, pairs, wJ, wK, **call, tau=tau, density_weighted=1)
        Qmax = Q.max()
        prs = [(i, j) for i in range(ns) for j in range(i + 1) if Q[i, j] * Qmax >= tau]
        vis = cnt = 0
        for a, (i, j) in enumerate(prs):
            for (k, l) in prs[: a + 1]:
                qq = Q[i, j] * Q[k, l]
                if qq >= tau:
                    vis += 1
                    cnt += qq * W[i, j, k, l] >= tau
        assert st["quartets_visited"] == vis
        assert st["quartets_computed"] == cnt
