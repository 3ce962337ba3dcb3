"""ctypes wrapper of the CPU oracle (oracle/oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package's library or binding.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "oracle.c")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (+OpenMP)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _SO, _SRC, "-lm"]
        )
    return _SO


class Options(C.Structure):
    _fields_ = [("tau", C.c_double), ("density_weighted", C.c_int32), ("sample_mod", C.c_uint32), ("sample_seed", C.c_uint32)]


class Stats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("pairs_total", "pairs_kept", "quartets_visited", "quartets_computed", "prim_quartets")]

    def asdict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
    return _lib


def _sys_args(sysm):
    xyz = np.ascontiguousarray(sysm.xyz, dtype=np.float64)
    sh = np.ascontiguousarray(sysm.shells, dtype=np.int32)
    ex = np.ascontiguousarray(sysm.exps, dtype=np.float64)
    co = np.ascontiguousarray(sysm.coefs, dtype=np.float64)
    keep = (xyz, sh, ex, co)
    args = (
        C.c_int(xyz.shape[0]), xyz.ctypes.data_as(C.c_void_p), C.c_int(sh.shape[0]), sh.ctypes.data_as(C.c_void_p),
        C.c_int(ex.shape[0]), ex.ctypes.data_as(C.c_void_p), co.ctypes.data_as(C.c_void_p),
    )
    return args, keep


def _ncart(l):
    return (l + 1) * (l + 2) // 2


def boys(mmax: int, T: float) -> np.ndarray:
    out = np.zeros(mmax + 1)
    lib().orc_boys(C.c_int(mmax), C.c_double(T), out.ctypes.data_as(C.c_void_p))
    return out


def boys_op(mmax: int, T: float, rho: float, omega: float) -> np.ndarray:
    out = np.zeros(mmax + 1)
    lib().orc_boys_op(C.c_int(mmax), C.c_double(T), C.c_double(rho), C.c_double(omega), out.ctypes.data_as(C.c_void_p))
    return out


def eri_shell(sysm, i, j, k, l, omega=0.0, deriv=False):
    args, keep = _sys_args(sysm)
    ls = [int(sysm.shells[s, 1]) for s in (i, j, k, l)]
    shape = tuple(_ncart(x) for x in ls)
    out = np.zeros(shape)
    dout = np.zeros((4, 3) + shape) if deriv else None
    rc = lib().orc_eri_shell(*args, C.c_int(i), C.c_int(j), C.c_int(k), C.c_int(l), C.c_double(omega),
                             out.ctypes.data_as(C.c_void_p), dout.ctypes.data_as(C.c_void_p) if deriv else None)
    assert rc == 0, rc
    return (out, dout) if deriv else out


def eri_tensor(sysm, omega=0.0):
    args, keep = _sys_args(sysm)
    n = sysm.nbf
    out = np.zeros((n, n, n, n))
    rc = lib().orc_eri_tensor(*args, C.c_double(omega), out.ctypes.data_as(C.c_void_p))
    assert rc == 0, rc
    return out


def overlap(sysm):
    args, keep = _sys_args(sysm)
    n = sysm.nbf
    out = np.zeros((n, n))
    rc = lib().orc_overlap(*args, out.ctypes.data_as(C.c_void_p))
    assert rc == 0, rc
    return out


def schwarz(sysm):
    args, keep = _sys_args(sysm)
    n = sysm.nshell
    out = np.zeros((n, n))
    rc = lib().orc_schwarz(*args, out.ctypes.data_as(C.c_void_p))
    assert rc == 0, rc
    return out


def _mats(pairs):
    A = [np.ascontiguousarray(a, dtype=np.float64) for a, _ in pairs]
    B = [np.ascontiguousarray(b, dtype=np.float64) for _, b in pairs]
    PA = (C.c_void_p * len(A))(*[a.ctypes.data for a in A])
    PB = (C.c_void_p * len(B))(*[b.ctypes.data for b in B])
    return PA, PB, (A, B)


def _call(fn, sysm, pairs, wJ, wK, cJ, cK, cLR, omega, nout, tau=None, density_weighted=None, sample_mod=0, sample_seed=0):
    args, keep = _sys_args(sysm)
    PA, PB, keep2 = _mats(pairs)
    wJ = np.ascontiguousarray(wJ, dtype=np.float64)
    wK = np.ascontiguousarray(wK, dtype=np.float64)
    opt = Options(sysm.tau if tau is None else tau,
                  sysm.density_weighted if density_weighted is None else density_weighted, sample_mod, sample_seed)
    st = Stats()
    out = np.zeros(nout)
    rc = fn(*args, C.byref(opt), C.c_int(len(pairs)), PA, PB, wJ.ctypes.data_as(C.c_void_p), wK.ctypes.data_as(C.c_void_p),
            C.c_double(cJ), C.c_double(cK), C.c_double(cLR), C.c_double(omega), out.ctypes.data_as(C.c_void_p), C.byref(st))
    assert rc == 0, rc
    return out, st.asdict()


def gradient(sysm, pairs, wJ, wK, cJ, cK, cLR, omega, **kw):
    g, st = _call(lib().orc_gradient, sysm, pairs, wJ, wK, cJ, cK, cLR, omega, 3 * sysm.natom, **kw)
    return g.reshape(-1, 3), st


def energy(sysm, pairs, wJ, wK, cJ, cK, cLR, omega, **kw):
    e, st = _call(lib().orc_energy, sysm, pairs, wJ, wK, cJ, cK, cLR, omega, 1, **kw)
    return float(e[0]), st


def gradient_n4(sysm, pairs, wJ, wK, cJ, cK, cLR, omega):
    args, keep = _sys_args(sysm)
    PA, PB, keep2 = _mats(pairs)
    wJ = np.ascontiguousarray(wJ, dtype=np.float64)
    wK = np.ascontiguousarray(wK, dtype=np.float64)
    out = np.zeros(3 * sysm.natom)
    rc = lib().orc_gradient_n4(*args, C.c_int(len(pairs)), PA, PB, wJ.ctypes.data_as(C.c_void_p), wK.ctypes.data_as(C.c_void_p),
                               C.c_double(cJ), C.c_double(cK), C.c_double(cLR), C.c_double(omega), out.ctypes.data_as(C.c_void_p))
    assert rc == 0, rc
    return out.reshape(-1, 3)


def density_weights(sysm, pairs, wJ, wK, cJ, cK, cLR, want_W=True):
    """S9 quantities as the oracle's screening uses them: d[ns, ns] and (optionally) W[ns, ns, ns, ns]."""
    args, keep = _sys_args(sysm)
    PA, PB, keep2 = _mats(pairs)
    wJ = np.ascontiguousarray(wJ, dtype=np.float64)
    wK = np.ascontiguousarray(wK, dtype=np.float64)
    ns = sysm.nshell
    d = np.zeros((ns, ns))
    W = np.zeros((ns, ns, ns, ns)) if want_W else None
    rc = lib().orc_density_weights(*args, C.c_int(len(pairs)), PA, PB, wJ.ctypes.data_as(C.c_void_p), wK.ctypes.data_as(C.c_void_p),
                                   C.c_double(cJ), C.c_double(cK), C.c_double(cLR), d.ctypes.data_as(C.c_void_p),
                                   W.ctypes.data_as(C.c_void_p) if want_W else None)
    assert rc == 0, rc
    return d, W


def _fock_args(Bs, wJ, wK, wKT, n):
    B = [np.ascontiguousarray(b, dtype=np.float64) for b in Bs]
    F = [np.zeros((n, n)) for _ in B]
    PB = (C.c_void_p * len(B))(*[b.ctypes.data for b in B])
    PF = (C.c_void_p * len(F))(*[f.ctypes.data for f in F])
    w = [np.ascontiguousarray(x, dtype=np.float64) for x in (wJ, wK, wKT)]
    return B, F, PB, PF, w


def fock(sysm, Bs, wJ, wK, wKT, cK, cLR, omega, tau=None, density_weighted=None, sample_mod=0, sample_seed=0):
    """Fock-type matrices F_k = wJ_k J[B_k] - (cK K + cLR K_lr)[wK_k B_k + wKT_k B_k^T] (eqs 19, 34), unique-quartet loop."""
    args, keep = _sys_args(sysm)
    B, F, PB, PF, w = _fock_args(Bs, wJ, wK, wKT, sysm.nbf)
    opt = Options(sysm.tau if tau is None else tau, sysm.density_weighted if density_weighted is None else density_weighted,
                  sample_mod, sample_seed)
    st = Stats()
    rc = lib().orc_fock(*args, C.byref(opt), C.c_int(len(B)), PB, *[x.ctypes.data_as(C.c_void_p) for x in w],
                        C.c_double(cK), C.c_double(cLR), C.c_double(omega), PF, C.byref(st))
    assert rc == 0, rc
    return F, st.asdict()


def fock_n4(sysm, Bs, wJ, wK, wKT, cK, cLR, omega):
    """The same by the plain definition over all nshell^4 shell quartets (tiny inputs)."""
    args, keep = _sys_args(sysm)
    B, F, PB, PF, w = _fock_args(Bs, wJ, wK, wKT, sysm.nbf)
    rc = lib().orc_fock_n4(*args, C.c_int(len(B)), PB, *[x.ctypes.data_as(C.c_void_p) for x in w],
                           C.c_double(cK), C.c_double(cLR), C.c_double(omega), PF)
    assert rc == 0, rc
    return F


def sph_matrix(l: int) -> np.ndarray:
    """[2l+1 (l >= 2) or ncart(l), ncart(l)]: real solid harmonics m = -l..l over the normalised Cartesian components."""
    nc = _ncart(l)
    out = np.zeros((2 * l + 1 if l >= 2 else nc, nc))
    rc = lib().orc_sph_matrix(C.c_int(l), out.ctypes.data_as(C.c_void_p))
    assert rc == 0, rc
    return out


def sph_transform(sysm, flags) -> np.ndarray:
    """Block-diagonal C [nbf_in, nbf_cart] of the mixed input basis: flagged d/f shells spherical, the rest Cartesian."""
    blocks = [sph_matrix(int(l)) if (f and l >= 2) else np.eye(_ncart(int(l))) for l, f in zip(sysm.shells[:, 1], flags)]
    nin, nc = sum(b.shape[0] for b in blocks), sum(b.shape[1] for b in blocks)
    Cm = np.zeros((nin, nc))
    r = c = 0
    for b in blocks:
        Cm[r:r + b.shape[0], c:c + b.shape[1]] = b
        r += b.shape[0]; c += b.shape[1]
    return Cm


def _onee_in(sysm, Z, P=None, W=None):
    Z = np.ascontiguousarray(Z, dtype=np.float64)
    assert Z.shape == (sysm.natom,)
    n = sysm.nbf
    P = None if P is None else np.ascontiguousarray(P, dtype=np.float64)
    W = None if W is None else np.ascontiguousarray(W, dtype=np.float64)
    for M in (P, W):
        assert M is None or M.shape == (n, n)
    return Z, P, W


def onee_matrices(sysm, Z):
    """S, T (kinetic), V (nuclear attraction, charges Z[natom]) over the normalised Cartesian functions (NEXT-4)."""
    args, keep = _sys_args(sysm)
    Z, _, _ = _onee_in(sysm, Z)
    n = sysm.nbf
    S, T, V = np.zeros((n, n)), np.zeros((n, n)), np.zeros((n, n))
    rc = lib().orc_onee_matrices(*args, Z.ctypes.data_as(C.c_void_p), *[x.ctypes.data_as(C.c_void_p) for x in (S, T, V)])
    assert rc == 0, rc
    return S, T, V


def onee_energy(sysm, Z, P, W) -> float:
    """sum P (T + V) + sum W S + V_nuc."""
    args, keep = _sys_args(sysm)
    Z, P, W = _onee_in(sysm, Z, P, W)
    e = np.zeros(1)
    rc = lib().orc_onee_energy(*args, *[x.ctypes.data_as(C.c_void_p) for x in (Z, P, W, e)])
    assert rc == 0, rc
    return float(e[0])


def onee_gradient(sysm, Z, P, W) -> np.ndarray:
    """Terms 1-3 of eq 7: sum P dH^core + sum W dS + dV_nuc, [natom, 3]."""
    args, keep = _sys_args(sysm)
    Z, P, W = _onee_in(sysm, Z, P, W)
    g = np.zeros(3 * sysm.natom)
    rc = lib().orc_onee_gradient(*args, *[x.ctypes.data_as(C.c_void_p) for x in (Z, P, W, g)])
    assert rc == 0, rc
    return g.reshape(-1, 3)


def sample_keep(i, j, k, l, mod, seed) -> bool:
    return bool(lib().orc_sample_keep(C.c_int(i), C.c_int(j), C.c_int(k), C.c_int(l), C.c_uint32(mod), C.c_uint32(seed)))


def num_threads() -> int:
    return int(lib().orc_num_threads())
