"""ctypes binding of libtdgrad.so (include/tdgrad.h): argument marshalling only.

Every step of the path runs inside the CUDA library; there is no CPU fallback: importing works without the
library (so that workload generation can be used anywhere), but any call raises if ``libtdgrad.so`` is missing
or no CUDA device is present.  Never imports ``oracle``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtdgrad.so")
NCLASS = 55
_lib = None

SYMBOLS = ["tdg_create", "tdg_destroy", "tdg_set_system", "tdg_nbf", "tdg_set_spherical", "tdg_set_shard", "tdg_set_streams", "tdg_plan", "tdg_schwarz", "tdg_gradient",
           "tdg_energy", "tdg_fock", "tdg_onee_gradient", "tdg_rys", "tdg_rys_static", "tdg_fp64_peak", "tdg_strerror", "tdg_last_error"]


RYS_STATIC_MAX = 16384   # TDG_RYS_STATIC_MAX of include/tdgrad.h


class TdgError(RuntimeError):
    pass


class Options(C.Structure):
    _fields_ = [("tau", C.c_double), ("density_weighted", C.c_int32), ("sample_mod", C.c_uint32), ("sample_seed", C.c_uint32)]


class Stats(C.Structure):
    _fields_ = [("pairs_total", C.c_int64), ("pairs_kept", C.c_int64), ("quartets_visited", C.c_int64),
                ("quartets_computed", C.c_int64), ("prim_quartets", C.c_int64), ("quartets_by_class", C.c_int64 * NCLASS),
                ("prim_quartets_by_class", C.c_int64 * NCLASS),
                ("ms_by_class", C.c_float * NCLASS), ("ms_prepare", C.c_float), ("ms_total", C.c_float), ("launches", C.c_int32),
                ("groups", C.c_int32)]

    def asdict(self):
        d = {k: getattr(self, k) for k in ("pairs_total", "pairs_kept", "quartets_visited", "quartets_computed", "prim_quartets",
                                           "ms_prepare", "ms_total", "launches", "groups")}
        d["quartets_by_class"] = list(self.quartets_by_class)
        d["prim_quartets_by_class"] = list(self.prim_quartets_by_class)
        d["ms_by_class"] = list(self.ms_by_class)
        return d


def lib():
    """Load libtdgrad.so; raises (no fallback) when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            try:   # build the CUDA library in-tree (nvcc, ~10 min); this is the product itself, not a fallback
                from paper_2407_16586_b200 import build as _build

                _build.build()
            except Exception as exc:
                raise TdgError("libtdgrad.so is missing and could not be built (%s); there is no CPU fallback" % exc)
        L = C.CDLL(LIB_PATH)
        L.tdg_strerror.restype = C.c_char_p
        L.tdg_last_error.restype = C.c_char_p
        L.tdg_last_error.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def class_ls(cls: int):
    """(la, lb, lc, ld) of quartet class index cls = c1 (c1+1)/2 + c2 over pair classes c = la (la+1)/2 + lb."""
    pcs = [(la, lb) for la in range(4) for lb in range(la + 1)]
    c1 = 0
    while (c1 + 1) * (c1 + 2) // 2 <= cls:
        c1 += 1
    c2 = cls - c1 * (c1 + 1) // 2
    return pcs[c1] + pcs[c2]


def class_name(cls: int) -> str:
    s = "spdf"
    la, lb, lc, ld = class_ls(cls)
    return "(%s%s|%s%s)" % (s[la], s[lb], s[lc], s[ld])


def model_flops(cls: int, quartets: int, prim_quartets: int) -> float:
    """Algorithmic FP64 FLOPs of `quartets` contracted / `prim_quartets` primitive quartets of class `cls`
    (Rys-direct model of SURVEY.md 8(d) / DESIGN.md "Work per unit"; two operators)."""
    la, lb, lc, ld = class_ls(cls)
    L = la + lb + lc + ld
    nr = (L + 1) // 2 + 1
    nc = 1
    for l in (la, lb, lc, ld):
        nc *= (l + 1) * (l + 2) // 2
    c2d = 3 * (6 * (la + lb + 2) * (lc + ld + 2) + 2 * (la + 1) * (lb + 2) * (lc + 2) * (ld + 2)) + 27 * (la + 1) * (lb + 1) * (lc + 1) * (ld + 1)
    per_prim = 2 * nr * c2d + nc * nr * 90 + 2 * (60 + 20 * nr)
    return float(prim_quartets) * per_prim + float(quartets) * nc * 100


def _ptr(x):
    """Device/host address of a numpy array or a torch tensor."""
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


def shard_of_env():
    """(rank, world size) of this process under torchrun (RANK / WORLD_SIZE), else (0, 1)."""
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def allreduce_partial(partial, group=None):
    """Sum the per-rank partial gradients (torch tensor, in place) over the process group: the path's only exchange step."""
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(partial, op=dist.ReduceOp.SUM, group=group)
    return partial


class Context:
    """One tdg_ctx on one CUDA device."""

    def __init__(self, device: int = 0):
        self._h = C.c_void_p()
        rc = lib().tdg_create(C.byref(self._h), C.c_int(device))
        if rc != 0:
            self._h = C.c_void_p()
            raise TdgError("tdg_create(device=%d) failed: %s (no CPU fallback)" % (device, lib().tdg_strerror(rc).decode()))
        self.natom = 0
        self.nshell = 0

    def _check(self, rc, what):
        if rc != 0:
            raise TdgError("%s: %s [%s]" % (what, lib().tdg_strerror(rc).decode(), lib().tdg_last_error(self._h).decode()))

    def close(self):
        if self._h:
            lib().tdg_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_system(self, sysm):
        xyz = np.ascontiguousarray(sysm.xyz, dtype=np.float64)
        sh = np.ascontiguousarray(sysm.shells, dtype=np.int32)
        ex = np.ascontiguousarray(sysm.exps, dtype=np.float64)
        co = np.ascontiguousarray(sysm.coefs, dtype=np.float64)
        rc = lib().tdg_set_system(self._h, C.c_int(xyz.shape[0]), C.c_void_p(xyz.ctypes.data), C.c_int(sh.shape[0]),
                                  C.c_void_p(sh.ctypes.data), C.c_int(ex.shape[0]), C.c_void_p(ex.ctypes.data), C.c_void_p(co.ctypes.data))
        self._check(rc, "tdg_set_system")
        self.natom, self.nshell = int(xyz.shape[0]), int(sh.shape[0])

    def nbf(self) -> int:
        n = C.c_int()
        self._check(lib().tdg_nbf(self._h, C.byref(n)), "tdg_nbf")
        return n.value

    def set_spherical(self, flags=None):
        """flags[nshell] (nonzero: the d/f shell is spherical) or None for all Cartesian; see include/tdgrad.h."""
        if flags is None:
            rc = lib().tdg_set_spherical(self._h, None)
        else:
            f = np.ascontiguousarray(flags, dtype=np.int32)
            rc = lib().tdg_set_spherical(self._h, C.c_void_p(f.ctypes.data))
        self._check(rc, "tdg_set_spherical")

    def set_shard(self, rank: int, nranks: int):
        """This context computes the work items `rank` mod `nranks`; call before :meth:`plan`."""
        self._check(lib().tdg_set_shard(self._h, C.c_int(rank), C.c_int(nranks)), "tdg_set_shard")

    def set_streams(self, nstreams: int):
        """Deal the class launches of a call over `nstreams` CUDA streams (the caller's + internal ones)."""
        self._check(lib().tdg_set_streams(self._h, C.c_int(nstreams)), "tdg_set_streams")

    def plan(self, tau=0.0, density_weighted=0, sample_mod=0, sample_seed=0):
        opt = Options(tau, density_weighted, sample_mod, sample_seed)
        self._check(lib().tdg_plan(self._h, C.byref(opt)), "tdg_plan")

    def schwarz(self) -> np.ndarray:
        out = np.zeros((self.nshell, self.nshell))
        self._check(lib().tdg_schwarz(self._h, C.c_void_p(out.ctypes.data)), "tdg_schwarz")
        return out

    def gradient(self, pairs, wJ, wK, cJ, cK, cLR, omega, stream=None, out=None, want_stats=True):
        """pairs: list of (A, B), all numpy arrays (host) or all CUDA torch tensors (device), nbf x nbf float64 row-major.
        Returns (grad [natom,3] numpy or the given ``out`` tensor, stats dict or None)."""
        npair = len(pairs)
        on_dev = 0 if isinstance(pairs[0][0], np.ndarray) else 1
        keep = []
        if not on_dev:
            for a, b in pairs:
                keep.append((np.ascontiguousarray(a, dtype=np.float64), np.ascontiguousarray(b, dtype=np.float64)))
        else:
            for a, b in pairs:
                assert a.is_cuda and b.is_cuda and a.is_contiguous() and b.is_contiguous()
                keep.append((a, b))
        PA = (C.c_void_p * npair)(*[_ptr(a) for a, _ in keep])
        PB = (C.c_void_p * npair)(*[_ptr(b) for _, b in keep])
        wJ = np.ascontiguousarray(wJ, dtype=np.float64)
        wK = np.ascontiguousarray(wK, dtype=np.float64)
        st = Stats() if want_stats else None
        if out is None:
            g = np.zeros((self.natom, 3))
            gptr, g_dev = g.ctypes.data, 0
        else:
            g = out
            gptr, g_dev = out.data_ptr(), 1
        rc = lib().tdg_gradient(self._h, C.c_int(npair), PA, PB, C.c_int(on_dev), C.c_void_p(wJ.ctypes.data), C.c_void_p(wK.ctypes.data),
                                C.c_double(cJ), C.c_double(cK), C.c_double(cLR), C.c_double(omega),
                                C.c_void_p(stream if stream else 0), C.c_void_p(gptr), C.c_int(g_dev),
                                C.byref(st) if st is not None else None)
        self._check(rc, "tdg_gradient")
        return g, (st.asdict() if st is not None else None)

    def gradient_allreduce(self, pairs, wJ, wK, cJ, cK, cLR, omega, out, group=None, stream=None):
        """Sharded gradient: this rank's partial gradient from the CUDA kernels into the
        CUDA tensor ``out`` [natom, 3], then ONE all-reduce (sum) of its 3*natom doubles over ``group`` (NCCL when the
        tensors are on the GPU).  Requires :meth:`set_shard` (rank, world size) before :meth:`plan`.  No arithmetic here."""
        g, _ = self.gradient(pairs, wJ, wK, cJ, cK, cLR, omega, stream=stream, out=out, want_stats=False)
        return allreduce_partial(g, group)

    def energy(self, pairs, wJ, wK, cJ, cK, cLR, omega, stream=None) -> float:
        """Contracted energy E (host float) for the same arguments as :meth:`gradient` (untuned; for FD checks)."""
        npair = len(pairs)
        on_dev = 0 if isinstance(pairs[0][0], np.ndarray) else 1
        keep = [(np.ascontiguousarray(a, dtype=np.float64), np.ascontiguousarray(b, dtype=np.float64)) for a, b in pairs] if not on_dev else list(pairs)
        PA = (C.c_void_p * npair)(*[_ptr(a) for a, _ in keep])
        PB = (C.c_void_p * npair)(*[_ptr(b) for _, b in keep])
        wJ = np.ascontiguousarray(wJ, dtype=np.float64)
        wK = np.ascontiguousarray(wK, dtype=np.float64)
        e = C.c_double()
        rc = lib().tdg_energy(self._h, C.c_int(npair), PA, PB, C.c_int(on_dev), C.c_void_p(wJ.ctypes.data), C.c_void_p(wK.ctypes.data),
                              C.c_double(cJ), C.c_double(cK), C.c_double(cLR), C.c_double(omega), C.c_void_p(stream if stream else 0), C.byref(e))
        self._check(rc, "tdg_energy")
        return e.value

    def fock(self, Bs, wJ, wK, wKT, cK, cLR, omega, stream=None, out=None, want_stats=True):
        """Fock-type matrices F_k = wJ_k J[B_k] - (cK K + cLR K_lr)[wK_k B_k + wKT_k B_k^T] (include/tdgrad.h: tdg_fock).
        Bs: list of numpy arrays (host) or CUDA torch tensors; out: optional list of CUDA tensors to write into.
        Returns (list of F as numpy arrays, or ``out``; stats dict or None)."""
        nmat = len(Bs)
        on_dev = 0 if isinstance(Bs[0], np.ndarray) else 1
        keep = [np.ascontiguousarray(b, dtype=np.float64) for b in Bs] if not on_dev else list(Bs)
        n = self.nbf()
        if out is None:
            F = [np.zeros((n, n)) for _ in range(nmat)]
            f_dev = 0
        else:
            F, f_dev = out, 1
        PB = (C.c_void_p * nmat)(*[_ptr(b) for b in keep])
        PF = (C.c_void_p * nmat)(*[_ptr(f) for f in F])
        w = [np.ascontiguousarray(x, dtype=np.float64) for x in (wJ, wK, wKT)]
        st = Stats() if want_stats else None
        rc = lib().tdg_fock(self._h, C.c_int(nmat), PB, C.c_int(on_dev), *[C.c_void_p(x.ctypes.data) for x in w], C.c_double(cK), C.c_double(cLR),
                            C.c_double(omega), C.c_void_p(stream if stream else 0), PF, C.c_int(f_dev), C.byref(st) if st is not None else None)
        self._check(rc, "tdg_fock")
        return F, (st.asdict() if st is not None else None)

    def onee_gradient(self, Z, P, W, stream=None, out=None):
        """One-electron terms sum P d(T+V) + sum W dS + dV_nuc (include/tdgrad.h: tdg_onee_gradient).  Z: nuclear charges [natom];
        P, W: numpy arrays (host) or CUDA torch tensors (or None = zero).  Returns (gradient [natom, 3] as numpy array or ``out``, ms)."""
        Z = np.ascontiguousarray(Z, dtype=np.float64)
        mats = [m for m in (P, W) if m is not None]
        on_dev = 0 if (not mats or isinstance(mats[0], np.ndarray)) else 1
        keep = [None if m is None else (np.ascontiguousarray(m, dtype=np.float64) if not on_dev else m) for m in (P, W)]
        g = np.zeros((self.natom, 3)) if out is None else out
        ms = C.c_float()
        rc = lib().tdg_onee_gradient(self._h, C.c_void_p(Z.ctypes.data), *[C.c_void_p(_ptr(m)) if m is not None else None for m in keep],
                                     C.c_int(on_dev), C.c_void_p(stream if stream else 0), C.c_void_p(_ptr(g)), C.c_int(0 if out is None else 1),
                                     C.byref(ms))
        self._check(rc, "tdg_onee_gradient")
        return g, ms.value

    def rys(self, n, T, rho=None, omega=0.0) -> np.ndarray:
        T = np.ascontiguousarray(T, dtype=np.float64)
        rho = np.ones_like(T) if rho is None else np.ascontiguousarray(rho, dtype=np.float64)
        out = np.zeros((T.shape[0], 2 * n))
        rc = lib().tdg_rys(self._h, C.c_int(n), C.c_int(T.shape[0]), C.c_void_p(T.ctypes.data), C.c_void_p(rho.ctypes.data),
                           C.c_double(omega), C.c_void_p(out.ctypes.data))
        self._check(rc, "tdg_rys")
        return out

    def rys_static(self, n, T, rho=None, omega=0.0, stream=None) -> np.ndarray:
        """tdg_rys without any allocation on the device (include/tdgrad.h: tdg_rys_static; at most RYS_STATIC_MAX evaluations per call)."""
        T = np.ascontiguousarray(T, dtype=np.float64)
        rho = np.ones_like(T) if rho is None else np.ascontiguousarray(rho, dtype=np.float64)
        out = np.zeros((T.shape[0], 2 * n))
        rc = lib().tdg_rys_static(self._h, C.c_int(n), C.c_int(T.shape[0]), C.c_void_p(T.ctypes.data), C.c_void_p(rho.ctypes.data),
                                  C.c_double(omega), C.c_void_p(stream if stream else 0), C.c_void_p(out.ctypes.data))
        self._check(rc, "tdg_rys_static")
        return out

    def fp64_peak(self, ms=300.0) -> float:
        v = C.c_double()
        self._check(lib().tdg_fp64_peak(self._h, C.c_double(ms), C.byref(v)), "tdg_fp64_peak")
        return v.value
