"""Pins for the oracle's one-electron terms (NEXT-4; eq 7 terms 1-3; 1-e terms on the CPU in the paper).

None of these re-use the oracle's one-electron recurrences: closed forms for s functions (overlap, kinetic, nuclear attraction via
erf), T = 1/2 sum_x d^2 S / dA_x dB_x by finite differences of the separately pinned overlap, V as the tight-charge limit of the
separately pinned two-electron integrals, mpmath differentiation of the s-s closed forms for p and d functions, hydrogen-like
expectation values, the gradient against central finite differences of the energy, and translational invariance."""
import math

import mpmath as mp
import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl
from tests.helpers import tiny_system, two_centre_spdf_system

XYZ3 = np.array([[0.0, 0.0, 0.0], [1.3, 0.2, -0.4], [-0.5, 1.6, 0.7]])


def nprim(z, l):
    lx, ly, lz = l
    df = lambda n: math.prod(range(n, 0, -2)) if n > 0 else 1
    return (2 * z / math.pi) ** 0.75 * (4 * z) ** ((lx + ly + lz) / 2) / math.sqrt(df(2 * lx - 1) * df(2 * ly - 1) * df(2 * lz - 1))


def comps(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def F0(T):
    return 1.0 if T < 1e-14 else 0.5 * math.sqrt(math.pi / T) * math.erf(math.sqrt(T))


def test_s_functions_closed_forms(orc):
    """<a|b> = (pi/p)^{3/2} e^{-mu R^2};  <a|T|b> = mu (3 - 2 mu R^2) <a|b>;  <a|1/r_C|b> = (2 pi/p) e^{-mu R^2} F_0(p |P-C|^2)."""
    za, zb = 0.9, 0.35
    s = wl.make_custom_system(XYZ3, [[(0, [za], [1.0])], [(0, [zb], [1.0])], []])
    Z = np.array([1.5, 0.0, 2.5])
    S, T, V = orc.onee_matrices(s, Z)
    A, B = XYZ3[0], XYZ3[1]
    p, mu = za + zb, za * zb / (za + zb)
    R2 = float(np.sum((A - B) ** 2))
    nn = nprim(za, (0, 0, 0)) * nprim(zb, (0, 0, 0))
    s_ab = nn * (math.pi / p) ** 1.5 * math.exp(-mu * R2)
    assert S[0, 1] == pytest.approx(s_ab, rel=1e-14)
    assert S[0, 0] == pytest.approx(1.0, rel=1e-14)
    assert T[0, 1] == pytest.approx(mu * (3 - 2 * mu * R2) * s_ab, rel=1e-13)
    assert T[0, 0] == pytest.approx(1.5 * za, rel=1e-13)          # <T> of a normalised s Gaussian
    Pc = (za * A + zb * B) / p
    v = -sum(Z[c] * nn * 2 * math.pi / p * math.exp(-mu * R2) * F0(p * float(np.sum((Pc - XYZ3[c]) ** 2))) for c in range(3))
    assert V[0, 1] == pytest.approx(v, rel=1e-13)
    # one-centre: <V> = -Z 2 sqrt(2 zeta/pi) for the nucleus under the function
    s1 = wl.make_custom_system(XYZ3[:1], [[(0, [za], [1.0])]])
    _, _, V1 = orc.onee_matrices(s1, np.array([3.0]))
    assert V1[0, 0] == pytest.approx(-3.0 * 2 * math.sqrt(2 * za / math.pi), rel=1e-13)


def _ss_closed_mp(kind, a, b, A, B, Cn):
    """Unnormalised s-s overlap / kinetic / attraction (unit charge at Cn) as mpmath expressions of the centres."""
    p, mu = a + b, a * b / (a + b)
    R2 = sum((A[i] - B[i]) ** 2 for i in range(3))
    sab = (mp.pi / p) ** (mp.mpf(3) / 2) * mp.exp(-mu * R2)
    if kind == "S":
        return sab
    if kind == "T":
        return mu * (3 - 2 * mu * R2) * sab
    P = [(a * A[i] + b * B[i]) / p for i in range(3)]
    PC2 = sum((P[i] - Cn[i]) ** 2 for i in range(3))
    return -2 * mp.pi / p * mp.exp(-mu * R2) * mp.hyp1f1(mp.mpf(1) / 2, mp.mpf(3) / 2, -p * PC2)


def _raised_mp(kind, a, b, la, lb, A, B, Cn):
    """Integral over x^la.. e^{-a r_A^2} and x^lb.. e^{-b r_B^2} from the s-s closed form: a monomial times a Gaussian is a
    combination of centre derivatives of the Gaussian.  Uses (x-A)^n e^{-a(x-A)^2} built by the operator recursion
    g_{n+1} = (1/2a)(d/dA g_n + n g_{n-1}) evaluated by numerical differentiation in high precision."""
    def f(*c):
        return _ss_closed_mp(kind, a, b, c[0:3], c[3:6], Cn)

    # polynomial-in-derivative representation: g_n = sum_k c_k d^k/dA^k, built symbolically per direction
    def coeffs(n, z):
        # returns list c[k] with x^n e^{-z x^2} = sum_k c[k] (d/dA)^k e^{-z x^2}  (x = r - A); d/dA e = 2 z x e
        # recursion: x * (d^k e) = (1/2z) [ d^{k+1} e ] - ... is awkward; use Hermite relation instead:
        # d^k/dA^k e^{-z x^2} = z^{k/2} H_k(sqrt(z) x) e^{-z x^2}; invert monomials into Hermite polynomials.
        # x^n = sum_k inv[n][k] H_k(sqrt(z) x) z^{-n/2}
        import numpy.polynomial.hermite as H
        he = H.poly2herm([0] * n + [1])           # t^n in physicists' Hermite series of t = sqrt(z) x
        return [float(he[k]) * z ** (-n / 2) * z ** (-k / 2) for k in range(len(he))]

    ca = [coeffs(la[d], float(a)) for d in range(3)]
    cb = [coeffs(lb[d], float(b)) for d in range(3)]
    x0 = [mp.mpf(v) for v in list(A) + list(B)]
    total = mp.mpf(0)
    for kx in range(len(ca[0])):
        for ky in range(len(ca[1])):
            for kz in range(len(ca[2])):
                for jx in range(len(cb[0])):
                    for jy in range(len(cb[1])):
                        for jz in range(len(cb[2])):
                            co = ca[0][kx] * ca[1][ky] * ca[2][kz] * cb[0][jx] * cb[1][jy] * cb[2][jz]
                            if co == 0.0:
                                continue
                            order = (kx, ky, kz, jx, jy, jz)
                            val = f(*x0) if sum(order) == 0 else mp.diff(f, tuple(x0), order)
                            total += co * val
    return total


@pytest.mark.parametrize("la,lb", [(1, 0), (1, 1), (2, 1), (2, 2)])
def test_p_d_functions_vs_mpmath_derivatives_of_closed_forms(orc, la, lb):
    """S, T, V for p and d functions: monomial x Gaussian = Hermite combination of centre derivatives of the s-s closed forms,
    differentiated numerically by mpmath at 40 digits (no recurrence of the oracle involved)."""
    mp.mp.dps = 40
    za, zb = 0.8, 0.45
    s = wl.make_custom_system(XYZ3, [[(la, [za], [1.0])], [(lb, [zb], [1.0])], []])
    Z = np.array([0.0, 0.0, 1.0])
    S, T, V = orc.onee_matrices(s, Z)
    na = len(comps(la))
    picks = [(0, 0), (len(comps(la)) - 1, len(comps(lb)) - 1), (min(1, na - 1), 0)]
    for ia, ib in picks:
        ca, cb = comps(la)[ia], comps(lb)[ib]
        nn = nprim(za, ca) * nprim(zb, cb)
        for kind, M in (("S", S), ("T", T), ("V", V)):
            ref = float(_raised_mp(kind, mp.mpf(za), mp.mpf(zb), ca, cb, XYZ3[0], XYZ3[1], [mp.mpf(v) for v in XYZ3[2]])) * nn
            assert M[ia, na + ib] == pytest.approx(ref, rel=1e-10, abs=1e-13), (kind, ca, cb)


def test_overlap_matches_pinned_overlap_and_symmetry(orc):
    s = two_centre_spdf_system()
    Z = np.array([8.0, 1.0])
    S, T, V = orc.onee_matrices(s, Z)
    assert np.max(np.abs(S - orc.overlap(s))) < 1e-14
    for M in (S, T, V):
        assert np.max(np.abs(M - M.T)) < 1e-12
    assert np.all(np.linalg.eigvalsh(T) > 0)          # kinetic energy is positive definite
    assert np.all(np.linalg.eigvalsh(V) < 0)          # attraction by positive charges is negative definite


def test_kinetic_is_half_the_mixed_second_derivative_of_the_overlap(orc):
    """<grad m|grad n> = sum_x d^2 S_mn / dA_x dB_x (the functions depend on r - A, r - B), so T = 1/2 of it: second-order central
    differences of orc_overlap (pinned on its own) on a two-centre s/p/d/f system."""
    s0 = two_centre_spdf_system()
    _, T, _ = orc.onee_matrices(s0, np.zeros(2))
    nA = int(np.sum([wl.ncart(int(l)) for a, l in zip(s0.shells[:, 0], s0.shells[:, 1]) if a == 0]))
    h = 2e-3
    acc = np.zeros((nA, s0.nbf - nA))
    for x in range(3):
        tot = np.zeros_like(acc)
        for sa, sb in ((1, 1), (1, -1), (-1, 1), (-1, -1)):
            xyz = s0.xyz.copy()
            xyz[0, x] += sa * h
            xyz[1, x] += sb * h
            s = wl.make_custom_system(xyz, _shells_of(s0))
            tot += sa * sb * orc.overlap(s)[:nA, nA:]
        acc += tot / (4 * h * h)
    assert np.max(np.abs(0.5 * acc - T[:nA, nA:])) < 5e-6 * max(1.0, np.max(np.abs(T)))


def _shells_of(s):
    out = [[] for _ in range(s.natom)]
    for a, l, n, o in s.shells:
        out[a].append((int(l), s.exps[o:o + n], s.coefs[o:o + n]))
    return out


def test_attraction_is_the_tight_charge_limit_of_the_eri(orc):
    """-Z (mn|delta_C): a normalised s function of exponent g/2 squared is the unit charge (g/pi)^{3/2} e^{-g r^2}; for g -> inf the
    pinned two-electron integral (mn|ss) tends to <m|1/r_C|n> with relative error O(1/g)."""
    base = tiny_system(with_f=True)
    shells = _shells_of(base)
    g = 2.0e9
    xyz = np.vstack([base.xyz, [[0.4, -0.8, 0.3]]])
    probe = wl.make_custom_system(xyz, shells + [[(0, [g / 2], [1.0])]])
    Zq = 1.7
    _, _, V = orc.onee_matrices(wl.make_custom_system(xyz, shells + [[]]), np.array([0.0, 0.0, 0.0, Zq]))
    off = base.shell_offsets()
    ks = probe.nshell - 1
    for i in range(base.nshell):
        for j in range(base.nshell):
            blk = orc.eri_shell(probe, i, j, ks, ks)[:, :, 0, 0]
            ref = -Zq * blk
            got = V[off[i]:off[i] + blk.shape[0], off[j]:off[j] + blk.shape[1]]
            assert np.max(np.abs(got - ref)) < 1e-8 * max(1.0, np.max(np.abs(ref)))


def test_hydrogen_like_expectation_values(orc):
    """Virial-type check on a one-centre STO-like contraction: E(zeta) = 3 zeta/2 - Z 2 sqrt(2 zeta/pi) for one s Gaussian is
    minimal at zeta = 8 Z^2 / (9 pi) with E = -4 Z^2 / (3 pi)."""
    Zc = 2.0
    z = 8 * Zc * Zc / (9 * math.pi)
    s = wl.make_custom_system(np.zeros((1, 3)), [[(0, [z], [1.0])]])
    P = np.ones((1, 1))
    assert orc.onee_energy(s, np.array([Zc]), P, np.zeros((1, 1))) == pytest.approx(-4 * Zc * Zc / (3 * math.pi), rel=1e-13)


def _rand_mats(n, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n, n)), rng.standard_normal((n, n))       # general, nonsymmetric


@pytest.mark.parametrize("with_f", [False, True])
def test_gradient_vs_finite_differences_of_the_energy(orc, with_f):
    s0 = tiny_system(with_f=with_f)
    Z = np.array([8.0, 1.0, 1.5])
    P, W = _rand_mats(s0.nbf, 3)
    g = orc.onee_gradient(s0, Z, P, W)
    h = 1e-4
    fd = np.zeros_like(g)
    for a in range(s0.natom):
        for x in range(3):
            e = []
            for sg in (2, 1, -1, -2):
                xyz = s0.xyz.copy()
                xyz[a, x] += sg * h
                e.append(orc.onee_energy(wl.make_custom_system(xyz, _shells_of(s0)), Z, P, W))
            fd[a, x] = (-e[0] + 8 * e[1] - 8 * e[2] + e[3]) / (12 * h)
    assert np.max(np.abs(g - fd)) < 2e-8 * max(1.0, np.max(np.abs(g)))
    assert np.max(np.abs(g.sum(axis=0))) < 1e-10 * max(1.0, np.max(np.abs(g)))      # translational invariance


def test_gradient_terms_separately(orc):
    """Each of the three terms alone: W only (overlap derivative), P only with Z = 0 (kinetic), nuclear repulsion only."""
    s0 = two_centre_spdf_system()
    n = s0.nbf
    P, W = _rand_mats(n, 5)
    zero = np.zeros((n, n))
    Z0 = np.zeros(2)
    Z = np.array([3.0, 2.0])
    R = s0.xyz[0] - s0.xyz[1]
    r = np.linalg.norm(R)
    g_nuc = orc.onee_gradient(s0, Z, zero, zero)
    assert np.allclose(g_nuc[0], -Z[0] * Z[1] * R / r ** 3, rtol=1e-13) and np.allclose(g_nuc[1], -g_nuc[0], rtol=1e-13)

    def fd(Zv, Pv, Wv):
        h, out = 1e-4, np.zeros((2, 3))
        for a in range(2):
            for x in range(3):
                e = []
                for sg in (2, 1, -1, -2):
                    xyz = s0.xyz.copy()
                    xyz[a, x] += sg * h
                    e.append(orc.onee_energy(wl.make_custom_system(xyz, _shells_of(s0)), Zv, Pv, Wv))
                out[a, x] = (-e[0] + 8 * e[1] - 8 * e[2] + e[3]) / (12 * h)
        return out

    for Zv, Pv, Wv in ((Z0, zero, W), (Z0, P, zero), (Z, P, zero)):
        g = orc.onee_gradient(s0, Zv, Pv, Wv)
        ref = fd(Zv, Pv, Wv)
        assert np.max(np.abs(g - ref)) < 5e-8 * max(1.0, np.max(np.abs(g)))
        assert np.max(np.abs(g.sum(axis=0))) < 1e-9 * max(1.0, np.max(np.abs(g)))
