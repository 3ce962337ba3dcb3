"""Pins for the oracle's integrals (O1, O4-O7).  None of these re-use the oracle's recurrences:
closed form of (ss|ss), high-precision differentiation of that closed form for l>0, overlap
normalisation, operator limits, finite differences.  PAPER.md:52-58 (eqs 3-5), 236-253 (eqs 38-41)."""
import itertools
import math

import mpmath as mp
import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl

XYZ4 = np.array([[0.0, 0.0, 0.0], [1.3, 0.2, -0.4], [-0.5, 1.6, 0.7], [0.3, -0.9, 1.1]])
ZETA4 = [0.9, 0.5, 0.28, 2.0]


def one_prim_system(ls, zetas, xyz=XYZ4):
    return wl.make_custom_system(xyz, [[(l, [z], [1.0])] for l, z in zip(ls, zetas)])


def F0_mp(T):
    return mp.hyp1f1(mp.mpf(1) / 2, mp.mpf(3) / 2, -T)


def ssss_mp(a, b, c, d, A, B, C, D, omega=None):
    """Unnormalised primitive [ss|ss], closed form; omega: erf(omega r)/r."""
    p, q = a + b, c + d
    P = [(a * A[i] + b * B[i]) / p for i in range(3)]
    Q = [(c * C[i] + d * D[i]) / q for i in range(3)]
    AB2 = sum((A[i] - B[i]) ** 2 for i in range(3))
    CD2 = sum((C[i] - D[i]) ** 2 for i in range(3))
    PQ2 = sum((P[i] - Q[i]) ** 2 for i in range(3))
    rho = p * q / (p + q)
    pref = 2 * mp.pi ** (mp.mpf(5) / 2) / (p * q * mp.sqrt(p + q)) * mp.exp(-a * b / p * AB2 - c * d / q * CD2)
    if omega is None:
        return pref * F0_mp(rho * PQ2)
    s2 = mp.mpf(omega) ** 2 / (mp.mpf(omega) ** 2 + rho)
    return pref * mp.sqrt(s2) * F0_mp(s2 * rho * PQ2)


def nprim(z, l):
    lx, ly, lz = l
    df = lambda n: math.prod(range(n, 0, -2)) if n > 0 else 1
    L = lx + ly + lz
    return (2 * z / math.pi) ** 0.75 * (4 * z) ** (L / 2) / math.sqrt(df(2 * lx - 1) * df(2 * ly - 1) * df(2 * lz - 1))


def comps(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def test_component_order():
    assert comps(1) == [(1, 0, 0), (0, 1, 0), (0, 0, 1)]
    assert comps(2) == [(2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]
    assert comps(3)[:4] == [(3, 0, 0), (2, 1, 0), (2, 0, 1), (1, 2, 0)] and comps(3)[-1] == (0, 0, 3)


@pytest.mark.parametrize("omega", [None, 0.3, 2.0])
def test_ssss_closed_form(orc, omega):
    mp.mp.dps = 30
    s = one_prim_system([0, 0, 0, 0], ZETA4)
    for perm in [(0, 1, 2, 3), (0, 1, 2, 0), (0, 0, 0, 0), (3, 1, 1, 2)]:
        z = [ZETA4[i] for i in perm]
        ref = ssss_mp(*[mp.mpf(x) for x in z], *[[mp.mpf(v) for v in XYZ4[i]] for i in perm], omega=omega)
        ref = float(ref) * math.prod(nprim(x, (0, 0, 0)) for x in z)
        got = orc.eri_shell(s, *perm, omega=0.0 if omega is None else omega)
        assert got.ravel()[0] == pytest.approx(ref, rel=2e-14)


def test_golden_survey_crosscheck(orc):
    """tests/golden/ssss_crosscheck.txt: values quoted in SURVEY.md section 8(c) (survey-time throw-away
    McMurchie-Davidson script, non-authoritative; an early-warning for convention mismatches)."""
    import os

    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "ssss_crosscheck.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                vals[k] = float(v)
    s = one_prim_system([0, 0, 0, 0], ZETA4)
    v, dv = orc.eri_shell(s, 0, 1, 2, 3, deriv=True)
    vl, dvl = orc.eri_shell(s, 0, 1, 2, 3, omega=0.3, deriv=True)
    assert dv[0, 0].ravel()[0] == pytest.approx(vals["dAx_full_0123"], rel=1e-11)
    assert dvl[0, 0].ravel()[0] == pytest.approx(vals["dAx_lr_0123"], rel=1e-11)
    # "with the fourth function on atom 0 instead": zeta = 2.0 moved to the position of atom 0
    s2 = one_prim_system([0, 0, 0, 0], ZETA4, xyz=np.array([XYZ4[0], XYZ4[1], XYZ4[2], XYZ4[0]]))
    assert orc.eri_shell(s2, 0, 1, 2, 3).ravel()[0] == pytest.approx(vals["ssss_full_0120"], rel=1e-12)
    assert orc.eri_shell(s2, 0, 1, 2, 3, omega=0.3).ravel()[0] == pytest.approx(vals["ssss_lr_0120"], rel=1e-12)


def test_one_centre_ssss_and_unit_overlap(orc):
    for z in (0.3, 1.0, 7.5):
        s = one_prim_system([0], [z], xyz=np.zeros((1, 3)))
        assert orc.eri_shell(s, 0, 0, 0, 0).ravel()[0] == pytest.approx(2 * math.sqrt(z / math.pi), rel=1e-14)
    for cfg in (0, 2):
        s = wl.make_system(cfg) if cfg == 0 else None
        if s is None:
            full = wl.make_system(2)  # take the first water only (has the f shell)
            keep = full.shells[:, 0] < 3
            s = wl.System(full.xyz[:3], full.shells[keep], full.exps, full.coefs)
        S = orc.overlap(s)
        assert np.abs(np.diag(S) - 1.0).max() < 5e-15
        assert np.allclose(S, S.T, atol=1e-15)
        assert np.linalg.eigvalsh(S).min() > 0


def high_l_ref(ls, zs, centres, comp, omega):
    """Primitive integral of Cartesian components `comp` by differentiating the (ss|ss) closed form:
    with d = d/dA_x and x = x - A_x:  x e^{-z r^2} = d e/(2z);  x^2 e = (d^2 + 2z) e/(4 z^2);  x^3 e = (d^3 + 6 z d) e/(8 z^3)."""
    mp.mp.dps = 40
    z = [mp.mpf(x) for x in zs]
    base = [[mp.mpf(v) for v in c] for c in centres]
    # operator polynomial per (centre, direction): list of (derivative order, coefficient)
    def poly(n, zeta):
        if n == 0:
            return [(0, mp.mpf(1))]
        if n == 1:
            return [(1, 1 / (2 * zeta))]
        if n == 2:
            return [(2, 1 / (4 * zeta**2)), (0, 2 * zeta / (4 * zeta**2))]
        if n == 3:
            return [(3, 1 / (8 * zeta**3)), (1, 6 * zeta / (8 * zeta**3))]
        raise ValueError
    terms = [poly(comp[c][x], z[c]) for c in range(4) for x in range(3)]

    def f(*flat):
        cs = [list(flat[3 * c : 3 * c + 3]) for c in range(4)]
        return ssss_mp(*z, *cs, omega=omega)

    flat0 = [v for c in base for v in c]
    total = mp.mpf(0)
    for choice in itertools.product(*terms):
        orders = tuple(o for o, _ in choice)
        coef = mp.mpf(1)
        for _, cf in choice:
            coef *= cf
        total += coef * (mp.diff(f, tuple(flat0), orders) if any(orders) else f(*flat0))
    return total


@pytest.mark.parametrize(
    "ls,omega",
    [((1, 0, 0, 0), None), ((1, 1, 0, 0), 0.3), ((1, 0, 1, 1), None), ((2, 0, 1, 0), 0.3), ((2, 1, 0, 0), None),
     ((0, 2, 0, 1), None), ((3, 0, 0, 0), 0.3), ((1, 0, 3, 0), None), ((2, 0, 2, 0), 0.3)],
)
def test_high_l_vs_differentiated_closed_form(orc, ls, omega):
    zs = [1.1, 0.6, 0.45, 0.9]
    s = one_prim_system(ls, zs)
    got = orc.eri_shell(s, 0, 1, 2, 3, omega=0.0 if omega is None else omega)
    cl = [comps(l) for l in ls]
    rng = np.random.default_rng(sum(ls))
    idxs = list(itertools.product(*[range(len(c)) for c in cl]))
    picks = [idxs[i] for i in rng.choice(len(idxs), size=min(4, len(idxs)), replace=False)]
    for idx in picks:
        comp = [cl[c][idx[c]] for c in range(4)]
        ref = float(high_l_ref(ls, zs, XYZ4, comp, omega)) * math.prod(nprim(zs[c], comp[c]) for c in range(4))
        assert got[idx] == pytest.approx(ref, rel=1e-11, abs=1e-15), (idx, comp)


def test_two_centre_high_l_same_centre(orc):
    """Coincident centres (A=B, C=D), d and f functions: still the differentiated closed form."""
    ls, zs = (2, 1, 3, 0), [0.8, 1.4, 0.7, 0.5]
    xyz = np.array([XYZ4[0], XYZ4[0], XYZ4[2], XYZ4[2]])
    s = one_prim_system(ls, zs, xyz=xyz)
    got = orc.eri_shell(s, 0, 1, 2, 3)
    cl = [comps(l) for l in ls]
    for idx in [(0, 0, 0, 0), (4, 2, 7, 0), (5, 1, 9, 0)]:
        comp = [cl[c][idx[c]] for c in range(4)]
        ref = float(high_l_ref(ls, zs, xyz, comp, None)) * math.prod(nprim(zs[c], comp[c]) for c in range(4))
        assert got[idx] == pytest.approx(ref, rel=1e-11, abs=1e-15)


def test_omega_limits(orc):
    """omega -> infinity: erf integrals equal full Coulomb; omega -> 0: (mn|ls)_lr / omega -> (2/sqrt(pi)) S_mn S_ls."""
    from tests.helpers import tiny_system

    s = tiny_system(with_f=True)
    full = orc.eri_tensor(s)
    big = orc.eri_tensor(s, omega=1e6)
    assert np.abs(full - big).max() <= 1e-11 * np.abs(full).max()
    w = 1e-6
    small = orc.eri_tensor(s, omega=w) / w
    S = orc.overlap(s)
    ref = 2 / math.sqrt(math.pi) * np.einsum("mn,ls->mnls", S, S)
    assert np.abs(small - ref).max() <= 1e-9 * np.abs(ref).max()


def test_eri_permutational_symmetry(orc):
    from tests.helpers import tiny_system

    s = tiny_system(with_f=False)
    for om in (0.0, 0.3):
        g = orc.eri_tensor(s, omega=om)
        for perm in ("nmls", "mnsl", "lsmn", "slnm"):
            assert np.abs(g - np.einsum("mnls->" + perm, g)).max() < 1e-13


def _displaced(s, atom, x, h):
    xyz = s.xyz.copy()
    xyz[atom, x] += h
    return wl.System(xyz, s.shells, s.exps, s.coefs)


@pytest.mark.parametrize("om", [0.0, 0.3])
def test_derivative_integrals_vs_finite_difference(orc, om):
    """O7 (eq 39, 250 eq 40): centre derivatives vs Richardson-extrapolated central differences;
    sum over centres vanishes."""
    ls = (2, 1, 1, 3)
    s = wl.make_custom_system(XYZ4, [[(ls[0], [1.1, 0.4], [0.5, 0.6])], [(ls[1], [0.6], [1.0])],
                                     [(ls[2], [0.45, 1.3], [0.7, 0.2])], [(ls[3], [0.9], [1.0])]])
    v, dv = orc.eri_shell(s, 0, 1, 2, 3, omega=om, deriv=True)
    assert np.abs(dv.sum(axis=0)).max() < 1e-13 * max(1.0, np.abs(dv).max())
    scale = np.abs(dv).max()
    for c in range(4):
        for x in range(3):
            def fd(h):
                return (orc.eri_shell(_displaced(s, c, x, h), 0, 1, 2, 3, omega=om)
                        - orc.eri_shell(_displaced(s, c, x, -h), 0, 1, 2, 3, omega=om)) / (2 * h)
            h = 2e-3
            rich = (4 * fd(h / 2) - fd(h)) / 3
            assert np.abs(rich - dv[c, x]).max() < 2e-9 * scale, (c, x)
