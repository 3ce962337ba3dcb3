"""GPU parity of tdg_fock (Fock-type J/K build; eq 19, 197-207 eqs 33-34) against the
CPU oracle's orc_fock, element by element, through the C ABI.  Tolerance: max|dF| <= 1e-10 max|F| (FP64 atomics reorder the
sums; same norm-wise bar as the gradient, reading S13)."""
import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl
from tests.helpers import tiny_system, two_centre_spdf_system

pytestmark = pytest.mark.gpu
REL_TOL = 1e-10
EQ34 = dict(wJ=4.0, wK=1.0, wKT=1.0)       # sigma-vector build of the Z-vector iterations
EQ19 = dict(wJ=2.0, wK=1.0, wKT=0.0)       # Fock matrix of a (symmetric) difference density


@pytest.fixture(scope="module")
def ctx():
    from paper_2407_16586_b200 import tdgrad

    c = tdgrad.Context(0)
    yield c
    c.close()


def _cmp(F, R):
    for f, r in zip(F, R):
        d = np.abs(f - r).max()
        assert d <= REL_TOL * np.abs(r).max(), (d, np.abs(r).max())


def _both(ctx, orc, s, Bs, w, tau=None, dw=None, sample_mod=0, sample_seed=0, cK=wl.C_K, cLR=wl.C_LR, omega=wl.OMEGA):
    tau = s.tau if tau is None else tau
    dw = s.density_weighted if dw is None else dw
    wJ, wK, wKT = (np.array([x[k] for x in w]) for k in ("wJ", "wK", "wKT"))
    ctx.set_system(s)
    ctx.plan(tau, dw, sample_mod, sample_seed)
    F, st = ctx.fock(Bs, wJ, wK, wKT, cK, cLR, omega)
    R, rst = orc.fock(s, Bs, wJ, wK, wKT, cK, cLR, omega, tau=tau, density_weighted=dw, sample_mod=sample_mod, sample_seed=sample_seed)
    return F, st, R, rst


def _rand(n, seed, k):
    rng = np.random.default_rng(seed)
    return [rng.standard_normal((n, n)) for _ in range(k)]


@pytest.mark.parametrize("with_f", [False, True])
def test_fock_tiny_system(ctx, orc, with_f):
    s = tiny_system(with_f=with_f)
    B = _rand(s.nbf, 1, 3)
    B[1] = B[1] + B[1].T                                        # one symmetric input
    w = [EQ34, EQ19, dict(wJ=-0.7, wK=1.3, wKT=-0.4)]           # the last one needs the antisymmetric slot
    F, st, R, rst = _both(ctx, orc, s, B, w)
    _cmp(F, R)
    for k in ("pairs_kept", "quartets_visited", "quartets_computed", "prim_quartets"):
        assert st[k] == rst[k], k
    assert np.abs(F[0] - F[0].T).max() <= 1e-12 * np.abs(F[0]).max()   # eq 34 with wK = wKT gives a symmetric matrix


def test_fock_every_class_in_full(ctx, orc):
    s = two_centre_spdf_system()
    B = _rand(s.nbf, 2, 2)
    F, st, R, rst = _both(ctx, orc, s, B, [EQ34, dict(wJ=1.0, wK=0.9, wKT=0.2)])
    _cmp(F, R)
    assert all(c > 0 for c in st["quartets_by_class"])


def test_fock_switches(ctx, orc):
    s = tiny_system()
    B = _rand(s.nbf, 3, 1)
    for kw in (dict(cK=0.3, cLR=0.0, omega=0.0), dict(cK=0.0, cLR=0.0, omega=0.3), dict(cK=0.0, cLR=1.0, omega=0.7)):
        F, st, R, rst = _both(ctx, orc, s, B, [EQ34], **kw)
        _cmp(F, R)
    F, st, R, rst = _both(ctx, orc, s, B, [dict(wJ=0.0, wK=1.0, wKT=0.0)])   # exchange only, nonsymmetric result
    _cmp(F, R)


def test_fock_sigma_vector_contraction(ctx, orc):
    """sigma = C_v^T F~[C_v b C_o^T] C_o (eq 33) from the GPU matrix equals the oracle's."""
    s = wl.make_system(0)
    n = s.nbf
    rng = np.random.default_rng(5)
    q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    Co, Cv = q[:, :5], q[:, 5:]
    b = rng.standard_normal((n - 5, 5))
    Bm = Cv @ b @ Co.T
    F, st, R, rst = _both(ctx, orc, s, [Bm], [EQ34])
    sg, sr = Cv.T @ F[0] @ Co, Cv.T @ R[0] @ Co
    assert np.abs(sg - sr).max() <= REL_TOL * np.abs(sr).max()


def test_fock_cfg1_full_and_density_weighted(ctx, orc):
    s = wl.make_system(1)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(1))
    F, st, R, rst = _both(ctx, orc, s, [T, P], [EQ34, EQ19])
    _cmp(F, R)
    for k in ("pairs_kept", "quartets_visited", "quartets_computed", "prim_quartets"):
        assert st[k] == rst[k], k
    F, st, R, rst = _both(ctx, orc, s, [T, P], [EQ34, EQ19], tau=1e-8, dw=1)
    _cmp(F, R)
    assert st["quartets_visited"] == rst["quartets_visited"]
    assert abs(st["quartets_computed"] - rst["quartets_computed"]) <= 5
    assert st["quartets_computed"] < st["quartets_visited"]


def test_fock_cfg2_f_shells_subsample(ctx, orc):
    s = wl.make_system(2)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(2))
    F, st, R, rst = _both(ctx, orc, s, [T], [EQ34], sample_mod=1500, sample_seed=11)
    _cmp(F, R)
    assert st["quartets_computed"] == rst["quartets_computed"]


@pytest.mark.slow
def test_fock_cfg3_subsample(ctx, orc):
    s = wl.make_system(3)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(3))
    F, st, R, rst = _both(ctx, orc, s, [T], [EQ34], sample_mod=40000, sample_seed=3)
    _cmp(F, R)
    assert st["pairs_kept"] == rst["pairs_kept"]
    assert abs(st["quartets_computed"] - rst["quartets_computed"]) <= 3
