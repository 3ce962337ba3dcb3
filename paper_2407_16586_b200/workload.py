"""Seeded synthetic inputs (water clusters) for the ERI-derivative gradient path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library and
therefore holds none of the method's arithmetic: no integrals, no
normalisation, no screening.  It only lays out geometry, the synthetic basis
(raw exponents and raw contraction coefficients w.r.t. *normalised*
primitives) and random density matrices, following the recipe of
SURVEY.md §8(d) / DESIGN.md "Input recipe" (which stand in for the paper's
GFP + water / def2-SVP workload, PAPER.md:422, 438 — not in the container).

Conventions: bohr; shells are (atom, l, nprim, prim_off); Cartesian functions in
the order of DESIGN.md reading S7 (lx descending, then ly descending).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

ANGSTROM = 1.8897261246257702  # bohr per angstrom
BASE_SEED = 20240716

# Call parameters of every config (BASELINE.json): omegaB97X-like blending.
C_J = 1.0
C_K = 0.157706
C_LR = 0.842294
OMEGA = 0.3


def ncart(l: int) -> int:
    return (l + 1) * (l + 2) // 2


# (waters, extra f shell on O, tau, density_weighted)
CONFIGS = {
    0: dict(waters=1, f_shell=False, tau=0.0, density_weighted=0),
    1: dict(waters=8, f_shell=False, tau=1e-14, density_weighted=0),
    2: dict(waters=32, f_shell=True, tau=1e-12, density_weighted=0),
    3: dict(waters=256, f_shell=False, tau=1e-11, density_weighted=1),
    4: dict(waters=1024, f_shell=False, tau=1e-11, density_weighted=1),
}


@dataclass
class System:
    """Geometry + basis in the flat form both libraries take."""

    xyz: np.ndarray  # [natom,3] float64, bohr
    shells: np.ndarray  # [nshell,4] int32: atom, l, nprim, prim_off
    exps: np.ndarray  # [nprim_total] float64
    coefs: np.ndarray  # [nprim_total] float64 (w.r.t. normalised primitives)
    tau: float = 0.0
    density_weighted: int = 0
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def natom(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def nshell(self) -> int:
        return int(self.shells.shape[0])

    @property
    def nbf(self) -> int:
        return int(sum(ncart(int(l)) for l in self.shells[:, 1]))

    def shell_offsets(self) -> np.ndarray:
        n = np.array([ncart(int(l)) for l in self.shells[:, 1]], dtype=np.int64)
        return np.concatenate([[0], np.cumsum(n)])


def _element_basis(rng: np.random.Generator, f_shell: bool):
    """Synthetic basis tables: {element: [(l, exps, raw coefs)]}.

    Multi-primitive shells draw U(0.2,1) coefficients once per (element, shell),
    so every water shares one basis; single-primitive shells have coefficient 1.
    The draws are made in a fixed order (all O shells, then all H shells)
    regardless of ``f_shell`` so configs share the same numbers.
    """
    o_core = 5000.0 * 0.27 ** np.arange(6)
    c_o_s = rng.uniform(0.2, 1.0, 6)
    c_o_p = rng.uniform(0.2, 1.0, 3)
    c_h_s = rng.uniform(0.2, 1.0, 3)
    one = np.ones(1)
    O = [
        (0, o_core, c_o_s),
        (0, np.array([0.9]), one),
        (0, np.array([0.28]), one),
        (1, np.array([35.0, 7.9, 2.3]), c_o_p),
        (1, np.array([0.23]), one),
        (2, np.array([1.2]), one),
    ]
    if f_shell:
        O.append((3, np.array([0.8]), one))
    H = [
        (0, np.array([13.0, 2.0, 0.5]), c_h_s),
        (0, np.array([0.12]), one),
        (1, np.array([0.8]), one),
    ]
    return {"O": O, "H": H}


def _haar_rotation(rng: np.random.Generator) -> np.ndarray:
    g = rng.standard_normal((3, 3))
    q, r = np.linalg.qr(g)
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def water_cluster_xyz(n: int, rng: np.random.Generator) -> np.ndarray:
    """O,H,H,O,H,H,... coordinates in bohr."""
    mono = np.array(
        [
            [0.0, 0.0, 0.0],
            [0.96, 0.0, 0.0],
            [0.96 * np.cos(np.deg2rad(104.5)), 0.96 * np.sin(np.deg2rad(104.5)), 0.0],
        ]
    )
    if n == 1:
        return mono * ANGSTROM
    m = int(np.ceil(n ** (1.0 / 3.0) - 1e-9))
    sites = []
    for i in range(m):
        for j in range(m):
            for k in range(m):
                sites.append((i, j, k))
    sites = np.array(sites[:n], dtype=np.float64) * 3.1
    sites = sites + rng.uniform(-0.3, 0.3, sites.shape)
    out = np.empty((3 * n, 3))
    for w in range(n):
        rot = _haar_rotation(rng)
        out[3 * w : 3 * w + 3] = sites[w] + mono @ rot.T
    return out * ANGSTROM


def make_system(cfg: int) -> System:
    """Geometry + basis for BASELINE.json config ``cfg`` (0..4)."""
    c = CONFIGS[cfg]
    ss = np.random.SeedSequence(BASE_SEED + cfg)
    s_geom, _s_dens = ss.spawn(2)
    # One basis for every config (BASELINE.json: "same basis ... as config 0").
    basis = _element_basis(np.random.default_rng(np.random.SeedSequence(BASE_SEED).spawn(3)[2]), c["f_shell"])
    xyz = water_cluster_xyz(c["waters"], np.random.default_rng(s_geom))
    shells, exps, coefs = [], [], []
    off = 0
    for a in range(xyz.shape[0]):
        el = "O" if a % 3 == 0 else "H"
        for (l, e, d) in basis[el]:
            shells.append((a, l, len(e), off))
            exps.append(e)
            coefs.append(d)
            off += len(e)
    return System(
        xyz=np.ascontiguousarray(xyz),
        shells=np.array(shells, dtype=np.int32),
        exps=np.concatenate(exps),
        coefs=np.concatenate(coefs),
        tau=c["tau"],
        density_weighted=c["density_weighted"],
        name=f"cfg{cfg}-{c['waters']}w",
        meta=dict(cfg=cfg, **c),
    )


def make_custom_system(xyz_bohr, atom_shells, tau=0.0, density_weighted=0, name="custom") -> System:
    """Small hand-made systems for tests.

    ``atom_shells``: per atom, a list of (l, exps, coefs).
    """
    shells, exps, coefs = [], [], []
    off = 0
    for a, lst in enumerate(atom_shells):
        for (l, e, d) in lst:
            e = np.atleast_1d(np.asarray(e, dtype=np.float64))
            d = np.atleast_1d(np.asarray(d, dtype=np.float64))
            shells.append((a, l, len(e), off))
            exps.append(e)
            coefs.append(d)
            off += len(e)
    return System(
        xyz=np.ascontiguousarray(np.asarray(xyz_bohr, dtype=np.float64)),
        shells=np.array(shells, dtype=np.int32).reshape(-1, 4),
        exps=np.concatenate(exps),
        coefs=np.concatenate(coefs),
        tau=tau,
        density_weighted=density_weighted,
        name=name,
    )


def make_densities(nbf: int, seed, n_occ: int | None = None):
    """D = C_o C_o^T, random symmetric P with ||P||_F = ||D||_F, T = C_o X C_v^T (||X||_F = 1).

    numpy / CPU version (configs 0-2 and tests).  Returns float64 C-contiguous arrays.
    """
    rng = np.random.default_rng(seed)
    if n_occ is None:
        n_occ = max(1, nbf // 5)
    co, r = np.linalg.qr(rng.standard_normal((nbf, n_occ)))
    co = co * np.sign(np.diag(r))
    D = co @ co.T
    G = rng.standard_normal((nbf, nbf))
    S = 0.5 * (G + G.T)
    P = S * (np.sqrt(n_occ) / np.linalg.norm(S))
    G2 = rng.standard_normal((n_occ, nbf))
    Y = G2 - (G2 @ D)  # G (I - D): rows live in the virtual space
    T = co @ (Y / np.linalg.norm(Y))
    return (np.ascontiguousarray(D), np.ascontiguousarray(P), np.ascontiguousarray(T))


def make_densities_torch(nbf: int, seed: int, device, n_occ: int | None = None):
    """Same recipe with torch FP64 on ``device`` (configs 3-4: 328 MB / 5.2 GB per matrix).

    The numbers differ from :func:`make_densities` (different generator); whoever
    needs them on the host copies these tensors back, so oracle and CUDA path
    always see identical arrays.
    """
    import torch

    if n_occ is None:
        n_occ = max(1, nbf // 5)
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    f64 = torch.float64
    co, r = torch.linalg.qr(torch.randn((nbf, n_occ), generator=g, dtype=f64, device=device))
    co = co * torch.sign(torch.diagonal(r))
    del r
    D = co @ co.T
    D = 0.5 * (D + D.T)      # exactly symmetric whatever the GEMM's summation order (a rounding-level antisymmetric part would take a matrix slot)
    P = torch.randn((nbf, nbf), generator=g, dtype=f64, device=device)
    P = 0.5 * (P + P.T)
    P *= float(np.sqrt(n_occ)) / torch.linalg.norm(P)
    Y = torch.randn((n_occ, nbf), generator=g, dtype=f64, device=device)
    Y = Y - Y @ D
    Y /= torch.linalg.norm(Y)
    T = co @ Y
    return D.contiguous(), P.contiguous(), T.contiguous()


# ---- second workload: spatially decaying densities -------------------------------------------------
# Real TDDFT densities decay with distance, and "the pattern of nonzero elements in the density matrix" drives the cost of
# the ERI-derivative step.  The recipe below keeps the geometry, basis and call of a config and replaces the
# dense random matrices by ones whose elements fall off as exp(-r/DECAY_LENGTH) with the distance between the two atoms:
#   C[mu, o]   = g exp(-|R_mu - R_o| / L),   orbital o centred on the O atom of water (o mod n_waters), columns normalised
#   D          = C C^T,  scaled to ||D||_F = sqrt(n_occ)                       (localised "occupied" orbitals)
#   P[mu, nu]  = s exp(-|R_mu - R_nu| / L),  s symmetric Gaussian, scaled to ||P||_F = sqrt(n_occ)
#   T          = C Y,  Y[o, nu] = g exp(-|R_o - R_nu| / L),  scaled to ||T||_F = 1      (nonsymmetric, like C_o X C_v^T)
DECAY_LENGTH = 3.0  # bohr


def _bf_atoms(sysm: "System") -> np.ndarray:
    return np.concatenate([np.full(ncart(int(l)), int(a), dtype=np.int64) for a, l in zip(sysm.shells[:, 0], sysm.shells[:, 1])])


def make_decaying_densities(sysm: "System", seed, n_occ: int | None = None, length: float = DECAY_LENGTH):
    """numpy version (small systems); same distribution as :func:`make_decaying_densities_torch`."""
    nbf = sysm.nbf
    if n_occ is None:
        n_occ = max(1, nbf // 5)
    rng = np.random.default_rng(seed)
    at = _bf_atoms(sysm)
    R = sysm.xyz[at]                                                    # position of every basis function's atom
    heavy = np.array(sorted(set(int(a) for a, l in zip(sysm.shells[:, 0], sysm.shells[:, 1]) if l >= 2)) or sorted(set(at.tolist())))
    cen = sysm.xyz[heavy[np.arange(n_occ) % len(heavy)]]                # orbital centres
    dmo = np.linalg.norm(R[:, None, :] - cen[None, :, :], axis=2)       # [nbf, n_occ]
    dmm = np.linalg.norm(R[:, None, :] - R[None, :, :], axis=2)         # [nbf, nbf]
    C = rng.standard_normal((nbf, n_occ)) * np.exp(-dmo / length)
    C /= np.linalg.norm(C, axis=0, keepdims=True)
    D = C @ C.T
    D = 0.5 * (D + D.T)
    D *= np.sqrt(n_occ) / np.linalg.norm(D)
    S = rng.standard_normal((nbf, nbf))
    P = 0.5 * (S + S.T) * np.exp(-dmm / length)
    P *= np.sqrt(n_occ) / np.linalg.norm(P)
    Y = rng.standard_normal((n_occ, nbf)) * np.exp(-dmo.T / length)
    T = C @ Y
    T /= np.linalg.norm(T)
    return np.ascontiguousarray(D), np.ascontiguousarray(P), np.ascontiguousarray(T)


def make_decaying_densities_torch(sysm: "System", seed: int, device, n_occ: int | None = None, length: float = DECAY_LENGTH):
    """torch FP64 version on ``device`` for configs 3-4 (the same recipe; different generator, so different numbers)."""
    import torch

    nbf = sysm.nbf
    if n_occ is None:
        n_occ = max(1, nbf // 5)
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    f64 = torch.float64
    at = _bf_atoms(sysm)
    R = torch.as_tensor(sysm.xyz[at], dtype=f64, device=device)
    heavy = np.array(sorted(set(int(a) for a, l in zip(sysm.shells[:, 0], sysm.shells[:, 1]) if l >= 2)) or sorted(set(at.tolist())))
    cen = torch.as_tensor(sysm.xyz[heavy[np.arange(n_occ) % len(heavy)]], dtype=f64, device=device)
    dmo = torch.cdist(R, cen)
    C = torch.randn((nbf, n_occ), generator=g, dtype=f64, device=device) * torch.exp(-dmo / length)
    C /= torch.linalg.norm(C, dim=0, keepdim=True)
    D = C @ C.T
    D = 0.5 * (D + D.T)
    D *= float(np.sqrt(n_occ)) / torch.linalg.norm(D)
    S = torch.randn((nbf, nbf), generator=g, dtype=f64, device=device)
    P = 0.5 * (S + S.T)
    del S
    P *= torch.exp(-torch.cdist(R, R) / length)
    P *= float(np.sqrt(n_occ)) / torch.linalg.norm(P)
    Y = torch.randn((n_occ, nbf), generator=g, dtype=f64, device=device) * torch.exp(-dmo.T / length)
    T = C @ Y
    T /= torch.linalg.norm(T)
    return D.contiguous(), P.contiguous(), T.contiguous()


def density_seed(cfg: int) -> np.random.SeedSequence:
    return np.random.SeedSequence(BASE_SEED + cfg).spawn(2)[1]


def default_call(D, P, T):
    """The (A_k, B_k, wJ_k, wK_k) list of BASELINE.json: pairs (D,D),(D,P),(T,T), '2J-K' weights."""
    return [(D, D), (D, P), (T, T)], np.array([2.0, 2.0, 2.0]), np.array([1.0, 1.0, 1.0])
