"""GPU parity tests: libtdgrad (through the C ABI binding) against the CPU oracle, element by element.

Tolerance (BASELINE.json north_star; reading S13): max|dg| <= 1e-9 E_h/bohr and max|dg|/max|g| <= 1e-10.
Integer results (pair / quartet counts) must be identical.
"""
import os

import numpy as np
import pytest

from paper_2407_16586_b200 import workload as wl
from tests.helpers import CALL, densities, tiny_system, two_centre_spdf_system

pytestmark = pytest.mark.gpu

ABS_TOL = 1e-9
REL_TOL = 1e-10


@pytest.fixture(scope="module")
def ctx():
    from paper_2407_16586_b200 import tdgrad

    c = tdgrad.Context(0)
    yield c
    c.close()


@pytest.fixture(scope="module")
def cfg1_case(orc):
    """cfg 1 inputs and the oracle's full gradient, computed once for the tests that compare against it (24 s of oracle time each)."""
    s = wl.make_system(1)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(1))
    pairs, wJ, wK = wl.default_call(D, P, T)
    ref, rst = orc.gradient(s, pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"], tau=s.tau, density_weighted=s.density_weighted)
    return s, pairs, wJ, wK, ref, rst


def _run_gpu(ctx, s, pairs, wJ, wK, call=CALL):
    ctx.set_system(s)
    ctx.plan(s.tau, s.density_weighted)
    return ctx.gradient(pairs, wJ, wK, call["cJ"], call["cK"], call["cLR"], call["omega"])


def _compare(g, ref):
    d = np.max(np.abs(g - ref))
    assert d <= ABS_TOL, d
    assert d / np.max(np.abs(ref)) <= REL_TOL, d / np.max(np.abs(ref))


def _run_both(ctx, orc, s, pairs, wJ, wK, call=CALL, sample_mod=0, sample_seed=0, tau=None, dw=None):
    tau = s.tau if tau is None else tau
    dw = s.density_weighted if dw is None else dw
    ctx.set_system(s)
    ctx.plan(tau, dw, sample_mod, sample_seed)
    g, st = ctx.gradient(pairs, wJ, wK, call["cJ"], call["cK"], call["cLR"], call["omega"])
    ref, rst = orc.gradient(s, pairs, wJ, wK, call["cJ"], call["cK"], call["cLR"], call["omega"], tau=tau, density_weighted=dw,
                            sample_mod=sample_mod, sample_seed=sample_seed)
    return g, st, ref, rst


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7])
@pytest.mark.parametrize("omega", [0.0, 0.3, 5.0])
def test_rys_moments_vs_oracle_boys(ctx, orc, n, omega):
    """sum_r w_r x_r^k == G_k(T, rho, omega), k < 2n, with G the oracle's (attenuated) Boys vector (O2/O3, S8)."""
    rng = np.random.default_rng(n)
    T = np.concatenate([[0.0, 1e-7, 0.3, 1.0, 39.999, 40.0, 77.9, 78.0, 150.0, 3e4], rng.uniform(0, 90, 200), 10 ** rng.uniform(-6, 5, 50)])
    rho = rng.uniform(0.05, 50.0, T.shape[0])
    out = ctx.rys(n, T, rho, omega)
    for i in range(T.shape[0]):
        x, w = out[i, :n], out[i, n:]
        G = orc.boys_op(2 * n - 1, T[i], rho[i], omega) if omega > 0 else orc.boys(2 * n - 1, T[i])
        for k in range(2 * n):
            assert abs(np.sum(w * x ** k) - G[k]) <= 3e-13 * G[k], (n, omega, T[i], k)


@pytest.mark.parametrize("with_f", [False, True])
def test_schwarz_vs_oracle(ctx, orc, with_f):
    s = tiny_system(with_f=with_f)
    ctx.set_system(s)
    Q = ctx.schwarz()
    ref = orc.schwarz(s)
    assert np.max(np.abs(Q - ref) / ref) < 1e-12


def test_schwarz_cfg1(ctx, orc):
    s = wl.make_system(1)
    ctx.set_system(s)
    Q = ctx.schwarz()
    ref = orc.schwarz(s)
    big = ref > 1e-20
    assert np.max(np.abs(Q[big] - ref[big]) / ref[big]) < 1e-10
    assert np.max(np.abs(Q[~big] - ref[~big])) < 1e-20


@pytest.mark.parametrize("with_f", [False, True])
def test_tiny_system_all_classes(ctx, orc, with_f):
    s = tiny_system(with_f=with_f)
    D, P, T = densities(s.nbf)
    pairs, wJ, wK = wl.default_call(D, P, T)
    g, st, ref, rst = _run_both(ctx, orc, s, pairs, wJ, wK)
    _compare(g, ref)
    for k in ("pairs_total", "pairs_kept", "quartets_visited", "quartets_computed", "prim_quartets"):
        assert st[k] == rst[k], k


def test_two_centre_spdf_every_class_in_full(ctx, orc):
    """All 55 quartet classes, f shells on both centres, no screening, no subsample: every class kernel is compared on
    real two-centre quartets (the single f shell of tiny_system only gives the one-atom (ff|ff) the kernel skips)."""
    s = two_centre_spdf_system()
    D, P, T = densities(s.nbf, seed=13)
    pairs, wJ, wK = wl.default_call(D, P, T)
    g, st, ref, rst = _run_both(ctx, orc, s, pairs, wJ, wK)
    _compare(g, ref)
    for k in ("pairs_total", "pairs_kept", "quartets_visited", "quartets_computed", "prim_quartets"):
        assert st[k] == rst[k], k
    assert all(c > 0 for c in st["quartets_by_class"]), st["quartets_by_class"]
    # nonsymmetric pairs through the same classes
    rng = np.random.default_rng(8)
    M = [rng.standard_normal((s.nbf, s.nbf)) for _ in range(3)]
    pairs2 = [(M[0], M[1]), (M[2], M[2])]
    g, st, ref, rst = _run_both(ctx, orc, s, pairs2, np.array([0.9, -0.4]), np.array([0.6, 1.2]))
    _compare(g, ref)


def test_tiny_general_pairs_and_weights(ctx, orc):
    """Arbitrary nonsymmetric A != B pairs and weights exercise the sym/antisym split of the K term."""
    s = tiny_system(with_f=False)
    rng = np.random.default_rng(5)
    n = s.nbf
    M = [rng.standard_normal((n, n)) for _ in range(4)]
    pairs = [(M[0], M[1]), (M[2], M[2]), (M[3], M[0] + M[0].T)]
    wJ, wK = np.array([0.7, -1.3, 0.4]), np.array([1.1, 0.5, -0.8])
    g, st, ref, rst = _run_both(ctx, orc, s, pairs, wJ, wK)
    _compare(g, ref)


def test_tiny_no_lr_and_no_exchange(ctx, orc):
    s = tiny_system(with_f=False)
    D, P, T = densities(s.nbf)
    pairs, wJ, wK = wl.default_call(D, P, T)
    for call in (dict(cJ=1.0, cK=0.3, cLR=0.0, omega=0.0), dict(cJ=1.0, cK=0.0, cLR=0.0, omega=0.3), dict(cJ=0.0, cK=0.0, cLR=1.0, omega=0.7)):
        g, st, ref, rst = _run_both(ctx, orc, s, pairs, wJ, wK, call=call)
        _compare(g, ref)


def test_cfg0_golden_and_oracle(ctx, orc):
    import os

    s = wl.make_system(0)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(0))
    pairs, wJ, wK = wl.default_call(D, P, T)
    g, st, ref, rst = _run_both(ctx, orc, s, pairs, wJ, wK)
    _compare(g, ref)
    assert st["quartets_computed"] == rst["quartets_computed"] == 3081
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "cfg0_gradient.txt"))
    _compare(g, gold)
    assert np.max(np.abs(g.sum(axis=0))) < 1e-10


def test_cfg1_full(ctx, cfg1_case):
    s, pairs, wJ, wK, ref, rst = cfg1_case
    g, st = _run_gpu(ctx, s, pairs, wJ, wK)
    _compare(g, ref)
    for k in ("pairs_total", "pairs_kept", "quartets_visited", "quartets_computed", "prim_quartets"):
        assert st[k] == rst[k], (k, st[k], rst[k])


def test_cfg1_density_weighted_screening(ctx, orc):
    s = wl.make_system(1)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(1))
    pairs, wJ, wK = wl.default_call(D, P, T)
    g, st, ref, rst = _run_both(ctx, orc, s, pairs, wJ, wK, tau=1e-9, dw=1)
    _compare(g, ref)
    assert st["quartets_visited"] == rst["quartets_visited"]
    assert abs(st["quartets_computed"] - rst["quartets_computed"]) <= 5
    assert st["quartets_computed"] < st["quartets_visited"]


def test_cfg2_f_shells_subsample(ctx, orc):
    s = wl.make_system(2)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(2))
    pairs, wJ, wK = wl.default_call(D, P, T)
    g, st, ref, rst = _run_both(ctx, orc, s, pairs, wJ, wK, sample_mod=1500, sample_seed=11)
    _compare(g, ref)
    assert st["pairs_kept"] == rst["pairs_kept"]
    assert st["quartets_visited"] == rst["quartets_visited"]
    assert st["quartets_computed"] == rst["quartets_computed"]
    assert all(c > 0 for c in st["quartets_by_class"]), st["quartets_by_class"]   # the subsample hits all 55 classes


@pytest.mark.slow
def test_cfg3_subsample_bench_configuration(ctx, orc):
    """256 waters, the launch configuration bench.py times, on a deterministic subsample both sides evaluate (S12)."""
    s = wl.make_system(3)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(3))
    pairs, wJ, wK = wl.default_call(D, P, T)
    g, st, ref, rst = _run_both(ctx, orc, s, pairs, wJ, wK, sample_mod=40000, sample_seed=3)
    _compare(g, ref)
    assert st["pairs_kept"] == rst["pairs_kept"]
    assert abs(st["quartets_computed"] - rst["quartets_computed"]) <= 3


@pytest.mark.parametrize("with_f", [False, True])
def test_energy_vs_oracle(ctx, orc, with_f):
    s = tiny_system(with_f=with_f)
    D, P, T = densities(s.nbf)
    pairs, wJ, wK = wl.default_call(D, P, T)
    ctx.set_system(s)
    ctx.plan(0.0, 0)
    e = ctx.energy(pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    ref, _ = orc.energy(s, pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    assert abs(e - ref) <= 1e-11 * max(1.0, abs(ref)), (e, ref)


def test_energy_cfg1_screened(ctx, orc):
    s = wl.make_system(1)
    D, P, T = wl.make_densities(s.nbf, wl.density_seed(1))
    pairs, wJ, wK = wl.default_call(D, P, T)
    ctx.set_system(s)
    ctx.plan(s.tau, s.density_weighted)
    e = ctx.energy(pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    ref, _ = orc.energy(s, pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    assert abs(e - ref) <= 1e-10 * abs(ref), (e, ref)


def test_gpu_gradient_is_derivative_of_gpu_energy(ctx):
    """Central finite differences of tdg_energy (h = 1e-4 bohr) against tdg_gradient, all on the GPU."""
    import copy

    s = tiny_system(with_f=False)
    D, P, T = densities(s.nbf)
    pairs, wJ, wK = wl.default_call(D, P, T)
    args = (pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
    ctx.set_system(s)
    ctx.plan(0.0, 0)
    g, _ = ctx.gradient(*args)
    h = 1e-4
    for atom, x in ((0, 0), (1, 2), (2, 1)):
        e = []
        for sign in (+1, -1):
            s2 = copy.deepcopy(s)
            s2.xyz[atom, x] += sign * h
            ctx.set_system(s2)
            ctx.plan(0.0, 0)
            e.append(ctx.energy(*args))
        fd = (e[0] - e[1]) / (2 * h)
        assert abs(fd - g[atom, x]) <= 1e-6, (atom, x, fd, g[atom, x])


@pytest.mark.parametrize("nranks", [2, 3])
def test_sharded_work_items_partition_the_gradient(ctx, cfg1_case, nranks):
    """SURVEY.md 8(e) / PAPER.md:309: the rank shards (tdg_set_shard) partition the quartets exactly (integer counts add up
    to the unsharded ones, class by class) and their partial gradients sum to the oracle's gradient.  The shards run one
    after another on this GPU, each to completion; no rank waits on another."""
    s, pairs, wJ, wK, ref, _ = cfg1_case
    try:
        g_full, st_full = _run_gpu(ctx, s, pairs, wJ, wK)
        total = np.zeros_like(g_full)
        counts = {k: 0 for k in ("quartets_visited", "quartets_computed", "prim_quartets")}
        by_class = np.zeros(len(st_full["quartets_by_class"]), dtype=np.int64)
        for r in range(nranks):
            ctx.set_shard(r, nranks)
            ctx.plan(s.tau, s.density_weighted)
            g, st = ctx.gradient(pairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"])
            assert 0 < st["quartets_computed"] < st_full["quartets_computed"]
            assert st["quartets_computed"] < 1.5 * st_full["quartets_computed"] / nranks   # the deal balances
            total += g
            for k in counts:
                counts[k] += st[k]
            by_class += np.asarray(st["quartets_by_class"], dtype=np.int64)
        for k in counts:
            assert counts[k] == st_full[k], (k, counts[k], st_full[k])
        assert np.array_equal(by_class, np.asarray(st_full["quartets_by_class"], dtype=np.int64))
        _compare(total, ref)
        _compare(total, g_full)
    finally:
        ctx.set_shard(0, 1)


def test_set_shard_rejects_bad_arguments(ctx):
    from paper_2407_16586_b200 import tdgrad

    for rank, n in ((-1, 2), (2, 2), (0, 0)):
        with pytest.raises(tdgrad.TdgError):
            ctx.set_shard(rank, n)
    ctx.set_shard(0, 1)


@pytest.mark.slow
def test_cfg4_subsample_largest_configuration(ctx, orc):
    """1024 waters (25 600 bf, 21 GB packed densities): deterministic subsample both sides evaluate (S12).
    Last in the file: ~12 min, almost all of it the oracle's own Schwarz bounds over 7.5e7 shell pairs."""
    import torch

    s = wl.make_system(4)
    # densities generated on the device, as bench.py does for cfg 3-4 (the numpy recipe costs minutes of host GEMMs at 25 600 functions);
    # the CUDA path gets the device tensors, the oracle their host copies: both sides see identical arrays
    dev = wl.make_densities_torch(s.nbf, 20240716 + 4, "cuda")
    dpairs, wJ, wK = wl.default_call(*dev)
    hpairs, _, _ = wl.default_call(*[x.cpu().numpy() for x in dev])
    tau, dw, mod, seed = s.tau, s.density_weighted, 4000000, 4
    ctx.set_system(s)
    ctx.plan(tau, dw, mod, seed)
    out = torch.zeros((s.natom, 3), dtype=torch.float64, device="cuda")
    _, st = ctx.gradient(dpairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"], out=out)
    g = out.cpu().numpy()
    del dev, dpairs, out
    torch.cuda.empty_cache()
    ref, rst = orc.gradient(s, hpairs, wJ, wK, CALL["cJ"], CALL["cK"], CALL["cLR"], CALL["omega"], tau=tau, density_weighted=dw,
                            sample_mod=mod, sample_seed=seed)
    d = float(np.max(np.abs(g - ref)))
    print("cfg4 subsample: quartets gpu/oracle", st["quartets_computed"], rst["quartets_computed"], "pairs_kept", st["pairs_kept"], rst["pairs_kept"],
          "max|dg|", d, "max|g|", float(np.max(np.abs(ref))))
    _compare(g, ref)
    assert st["pairs_kept"] == rst["pairs_kept"]
    assert abs(st["quartets_computed"] - rst["quartets_computed"]) <= 3
