"""Pins for the oracle's real-solid-harmonic table (NEXT-2; PAPER.md:241 n_sph = 2l+1):
orthonormality under the oracle's own overlap integrals, harmonicity of the underlying polynomials (a homogeneous polynomial
of degree l is a solid harmonic iff its Laplacian vanishes: fixes the subspace), the textbook d functions, and invariance of a
spherical-basis trace under the Cartesian round trip."""
import itertools

import numpy as np

from paper_2407_16586_b200 import workload as wl


def _comps(l):
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


def _dfact(n):
    r = 1.0
    while n > 1:
        r *= n
        n -= 2
    return r


def test_one_centre_overlap_is_orthonormal(orc):
    xyz = np.array([[0.1, -0.2, 0.3]])
    atoms = [[(2, [1.3, 0.4], [0.6, 0.5]), (3, [0.9], [1.0]), (1, [0.7], [1.0]), (0, [0.5], [1.0])]]
    s = wl.make_custom_system(xyz, atoms)
    S = orc.overlap(s)
    C = orc.sph_transform(s, [1, 1, 1, 1])
    assert C.shape == (5 + 7 + 3 + 1, 6 + 10 + 3 + 1)
    Ssph = C @ S @ C.T
    assert np.abs(Ssph - np.eye(C.shape[0])).max() < 1e-13
    # the discarded combinations (s-type xx+yy+zz in d; three p-type in f) are orthogonal to the kept ones
    assert np.linalg.matrix_rank(C) == C.shape[0]


def test_polynomials_are_harmonic(orc):
    """Row m of C in unnormalised monomials, p(x,y,z) = sum_i C[m,i] / sqrt((2a-1)!!(2b-1)!!(2c-1)!!) x^a y^b z^c, satisfies
    Laplace's equation: checked exactly on the monomial coefficients."""
    for l in (2, 3):
        C = orc.sph_matrix(l)
        comps = _comps(l)
        for m in range(2 * l + 1):
            coef = {c: C[m, i] / np.sqrt(_dfact(2 * c[0] - 1) * _dfact(2 * c[1] - 1) * _dfact(2 * c[2] - 1)) for i, c in enumerate(comps)}
            lap = {}
            for (a, b, c), v in coef.items():
                for d, e in enumerate((a, b, c)):
                    if e >= 2:
                        key = [a, b, c]; key[d] -= 2
                        lap[tuple(key)] = lap.get(tuple(key), 0.0) + v * e * (e - 1)
            assert max([abs(x) for x in lap.values()] + [0.0]) < 1e-14, (l, m)
        # rows are linearly independent and mutually orthogonal under the component overlap (checked above with integrals)
        assert np.linalg.matrix_rank(C) == 2 * l + 1


def test_textbook_d_functions_and_f_constants(orc):
    C = orc.sph_matrix(2)   # Cartesian order xx, xy, xz, yy, yz, zz
    ref = np.array([[0, 1, 0, 0, 0, 0], [0, 0, 0, 0, 1, 0], [-0.5, 0, 0, -0.5, 0, 1], [0, 0, 1, 0, 0, 0],
                    [np.sqrt(3) / 2, 0, 0, -np.sqrt(3) / 2, 0, 0]])
    assert np.abs(C - ref).max() < 1e-15
    F = orc.sph_matrix(3)   # xxx, xxy, xxz, xyy, xyz, xzz, yyy, yyz, yzz, zzz
    assert abs(F[3, 9] - 1.0) < 1e-15 and abs(F[3, 2] + 3 / (2 * np.sqrt(5))) < 1e-15      # f_z3 = zzz - 3/(2 sqrt5)(xxz + yyz)
    assert abs(F[6, 0] - np.sqrt(5.0 / 8)) < 1e-15 and abs(F[6, 3] + 3 / (2 * np.sqrt(2))) < 1e-15
    assert abs(F[1, 4] - 1.0) < 1e-15
    assert np.abs(orc.sph_matrix(1) - np.eye(3)).max() == 0 and np.abs(orc.sph_matrix(0) - 1).max() == 0


def test_contraction_is_invariant_under_the_round_trip(orc):
    """E_sph = sum D_sph (pq|rs)_sph with (pq|rs)_sph = C C C C (mn|ls)  equals  E_cart with D_cart = C^T D_sph C."""
    from tests.helpers import tiny_system

    s = tiny_system(with_f=True)
    flags = [1] * s.nshell
    C = orc.sph_transform(s, flags)
    rng = np.random.default_rng(1)
    nin = C.shape[0]
    A, B = rng.standard_normal((nin, nin)), rng.standard_normal((nin, nin))
    g = orc.eri_tensor(s)
    gs = np.einsum("pm,qn,rl,ts,mnls->pqrt", C, C, C, C, g, optimize=True)
    e_sph = np.einsum("pq,rt,pqrt->", A, B, gs) - 0.3 * np.einsum("pr,qt,pqrt->", A, B, gs)
    Ac, Bc = C.T @ A @ C, C.T @ B @ C
    e_cart, _ = orc.energy(s, [(Ac, Bc)], np.ones(1), np.ones(1), 1.0, 0.3, 0.0, 0.3)
    assert abs(e_sph - e_cart) <= 1e-12 * abs(e_cart)
