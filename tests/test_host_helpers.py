"""CPU checks of the binding's host-side helpers (class indexing, the algorithmic FLOP model of DESIGN.md section 5) and of
the workload generator's bookkeeping (sizes of BASELINE.json's configs)."""
import numpy as np

from paper_2407_16586_b200 import tdgrad
from paper_2407_16586_b200 import workload as wl


def test_class_index_roundtrip_and_names():
    pcs = [(la, lb) for la in range(4) for lb in range(la + 1)]
    seen = set()
    for c1, (la, lb) in enumerate(pcs):
        for c2, (lc, ld) in enumerate(pcs[: c1 + 1]):
            cls = c1 * (c1 + 1) // 2 + c2
            assert tdgrad.class_ls(cls) == (la, lb, lc, ld)
            seen.add(cls)
    assert seen == set(range(tdgrad.NCLASS))
    assert tdgrad.class_name(0) == "(ss|ss)" and tdgrad.class_name(1) == "(ps|ss)" and tdgrad.class_name(54) == "(ff|ff)"
    # 21 classes for l <= 2
    assert sum(1 for c in range(55) if max(tdgrad.class_ls(c)) <= 2) == 21


def test_flop_model_matches_survey_examples():
    """SURVEY.md 8(d) quotes per-primitive-quartet examples: (ss|ss) ~0.5 k, (ps|ss) ~1.8 k, (pp|ps) ~11 k, (dd|dd) ~0.63 M."""
    def per_prim(la, lb, lc, ld):
        pcs = [(a, b) for a in range(4) for b in range(a + 1)]
        c1, c2 = pcs.index((la, lb)), pcs.index((lc, ld))
        return tdgrad.model_flops(c1 * (c1 + 1) // 2 + c2, 0, 1)
    assert 400 < per_prim(0, 0, 0, 0) < 600
    assert 1600 < per_prim(1, 0, 0, 0) < 2000
    assert 9e3 < per_prim(1, 1, 1, 0) < 13e3
    assert 5.5e5 < per_prim(2, 2, 2, 2) < 7e5
    # linear in both unit counts
    assert tdgrad.model_flops(1, 10, 40) == 10 * tdgrad.model_flops(1, 1, 0) + 40 * tdgrad.model_flops(1, 0, 1)


def test_config_sizes_match_baseline_json():
    expect = {0: (3, 12, 25), 1: (24, 96, 200), 2: (96, 416, 1120), 3: (768, 3072, 6400), 4: (3072, 12288, 25600)}
    for cfg, (natom, nshell, nbf) in expect.items():
        s = wl.make_system(cfg)
        assert (s.natom, s.nshell, s.nbf) == (natom, nshell, nbf)
    s0, s1 = wl.make_system(0), wl.make_system(1)
    assert np.array_equal(s0.exps[: s0.shells[-1, 3] + s0.shells[-1, 2]], s1.exps[: s0.shells[-1, 3] + s0.shells[-1, 2]])  # one basis for all


def test_default_call_weights():
    D = np.eye(3); P = 2 * np.eye(3); T = np.ones((3, 3))
    pairs, wJ, wK = wl.default_call(D, P, T)
    assert [(a is D, b is D) for a, b in pairs[:1]] == [(True, True)] and pairs[1][1] is P and pairs[2][0] is T
    assert list(wJ) == [2.0, 2.0, 2.0] and list(wK) == [1.0, 1.0, 1.0]


def test_decaying_density_recipe():
    """NEXT-4 workload: same norms as the dense recipe, elements fall off with the distance between the functions' atoms."""
    s = wl.make_system(1)
    D, P, T = wl.make_decaying_densities(s, 5)
    n_occ = s.nbf // 5
    assert abs(np.linalg.norm(D) - np.sqrt(n_occ)) < 1e-10 and abs(np.linalg.norm(P) - np.sqrt(n_occ)) < 1e-10
    assert abs(np.linalg.norm(T) - 1.0) < 1e-12
    assert np.array_equal(D, D.T) and np.array_equal(P, P.T) and np.abs(T - T.T).max() > 1e-3
    at = wl._bf_atoms(s)
    r = np.linalg.norm(s.xyz[at][:, None, :] - s.xyz[at][None, :, :], axis=2)
    near, far = np.abs(P[r < 2.0]).mean(), np.abs(P[r > 10.0]).mean()
    assert far < near * np.exp(-8.0 / wl.DECAY_LENGTH) * 3
    assert np.abs(D[r > 12.0]).max() < 0.05 * np.abs(D).max()


def test_build_role_count_matches_header_formula():
    """build.num_roles (one translation unit per class and role) against the cases stated in csrc/tdg_grad.cuh."""
    from paper_2407_16586_b200 import build

    assert build.num_roles(1, 0, 0, 0) == 1 and build.num_roles(1, 1, 1, 0) == 1
    assert build.num_roles(2, 1, 1, 0) == 2 and build.num_roles(2, 1, 2, 1) == 18 and build.num_roles(2, 2, 2, 1) == 12
    assert build.num_roles(2, 2, 2, 2) == 1 and build.num_roles(3, 0, 0, 0) == 1 and build.num_roles(3, 3, 3, 3) == 1
    assert build.num_roles(3, 1, 1, 0) == 4 and build.num_roles(3, 0, 1, 0) == 2 and build.num_roles(3, 2, 1, 0) == 7
    assert build.num_roles(3, 1, 1, 1) == 10 and build.num_roles(3, 1, 3, 0) == 15      # f classes: unrolled up to 15 roles
    assert build.num_roles(3, 2, 1, 1) == 1      # 20 roles: too many for an f class, block-per-quartet kernel


def test_bench_roofline_uses_the_capture_only_when_it_matches_the_build(monkeypatch):
    """bench.roofline_of: executed FLOPs come from the hash-stamped ncu capture under profiles/; a capture taken on other kernel
    sources, or on another workload (different per-class quartet count), gives null instead of a stale number."""
    import json
    import os
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    import bench
    from paper_2407_16586_b200 import ncu_classes, tdgrad

    cap = json.load(open(os.path.join(root, "profiles", "r02_ncu_classes_cfg3.json")))
    name = "(ps|ss)"
    top = [c for c in range(tdgrad.NCLASS) if tdgrad.class_name(c) == name][0]
    steps = 2
    ms, q, p = [0.0] * tdgrad.NCLASS, [0] * tdgrad.NCLASS, [0] * tdgrad.NCLASS
    ms[top] = 1300.0 * steps
    q[top] = cap["quartets_by_class"][name] * steps
    p[top] = cap["prim_quartets_by_class"][name] * steps
    monkeypatch.setattr(ncu_classes, "source_hash", lambda: cap["source_hash"])
    r = bench.roofline_of(ms, q, p, 9000.0 * steps, 34.2, 3, steps)
    assert r["kernel"].endswith(name) and r["capture_hash"] == cap["source_hash"]
    want = cap["classes"][name]["flops"] / 1.3 * 1e-12                      # executed FLOPs of one call / 1.3 s
    assert abs(r["achieved"] - want) < 1e-9 * want and abs(r["frac"] - want / 34.2) < 1e-12
    assert r["traffic"] == cap["classes"][name]["dram_read"] + cap["classes"][name]["dram_write"]
    assert 0.0 < r["frac"] < 1.0 and r["model_frac"] is not None
    # other kernel sources
    monkeypatch.setattr(ncu_classes, "source_hash", lambda: "0123456789abcdef")
    r2 = bench.roofline_of(ms, q, p, 9000.0 * steps, 34.2, 3, steps)
    assert r2["achieved"] is None and r2["frac"] is None and "older than the kernel sources" in r2["note"]
    # same sources, other workload
    monkeypatch.setattr(ncu_classes, "source_hash", lambda: cap["source_hash"])
    q[top] += 1
    r3 = bench.roofline_of(ms, q, p, 9000.0 * steps, 34.2, 3, steps)
    assert r3["frac"] is None and "different workload" in r3["note"]
