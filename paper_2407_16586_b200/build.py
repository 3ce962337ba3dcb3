"""Builds libtdgrad.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2407_16586_b200.build [--force]
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libtdgrad.so")
LMAX = 3
PAIR_CLASSES = [(la, lb) for la in range(LMAX + 1) for lb in range(la + 1)]
QUARTET_CLASSES = [p + q for i, p in enumerate(PAIR_CLASSES) for q in PAIR_CLASSES[: i + 1]]   # bra class >= ket class
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]
# per-class compile flags: minimum resident blocks per SM of __launch_bounds__ (registers traded for occupancy), measured on
# cfg 3 (profiles/r02_variants.md): class -> extra nvcc flags
CLASS_FLAGS: dict = {(0, 0, 0, 0): ["-DTDG_MINB=4", "-DTDG_DUAL_RYS=1"], (1, 0, 0, 0): ["-DTDG_MINB=3"], (2, 0, 0, 0): ["-DTDG_MINB=3"],
                     (1, 0, 1, 0): ["-DTDG_DUAL_RYS=1"]}   # TDG_DUAL_RYS: both operators' Rys rules evaluated back to back (tdg_grad.cuh)


MAX_ROLES_F = 15   # TDG_MAX_ROLES_F of csrc/tdg_grad.cuh


def ncart(l: int) -> int:
    return (l + 1) * (l + 2) // 2


def num_roles(la: int, lb: int, lc: int, ld: int) -> int:
    """QC<la,lb,lc,ld>::NROLE of csrc/tdg_grad.cuh (a static_assert in tdg_class.cu and the launcher table catch a mismatch)."""
    rc = 54 if (la, lb, lc, ld) == (2, 2, 2, 1) else 27
    nab, kdn = ncart(la) * ncart(lb), ncart(lc) * ncart(ld)
    abn1 = nab if rc // kdn >= nab else max(rc // kdn, 1)
    nrole1 = -(-nab // abn1)
    small = nab * kdn <= 27 or nrole1 <= (MAX_ROLES_F if 3 in (la, lb, lc, ld) else 18)
    return nrole1 if small else 1
DEPS = {   # headers each source includes
    "tdg_class.cu": ["tdg_common.cuh", "tdg_grad.cuh", "tdg_gradb.cuh", "tdg_fock.cuh", "rys_meta.inc"],
    "tdg_aux.cu": ["tdg_common.cuh", "tdg_internal.h", "rys_meta.inc", "rys_tables.inc", "boys_tables.inc"],
    "tdg_onee.cu": ["tdg_common.cuh", "tdg_internal.h", "rys_meta.inc"],
    "tdg_noalloc.cu": ["tdg_common.cuh", "tdg_internal.h", "rys_meta.inc"],
    "tdg_api.cu": ["tdg_common.cuh", "tdg_grad.cuh", "tdg_internal.h", "tdg_classes.inc", "rys_meta.inc", "../../include/tdgrad.h"],
}


def _newest_header(src: str) -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in DEPS[src])


def _compile(job):
    src, obj, extra = job
    cmd = [NVCC] + FLAGS + extra + ["-c", os.path.join(CSRC, src), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    with open(obj + ".cmd", "w") as f:   # an object is stale when its flags change, not only when its sources do
        f.write(" ".join(FLAGS + extra))
    return obj


def _same_flags(obj, extra) -> bool:
    try:
        return open(obj + ".cmd").read() == " ".join(FLAGS + extra)
    except OSError:
        return False


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    jobs = [("tdg_api.cu", os.path.join(OBJ, "tdg_api.o"), []), ("tdg_aux.cu", os.path.join(OBJ, "tdg_aux.o"), []),
            ("tdg_onee.cu", os.path.join(OBJ, "tdg_onee.o"), []), ("tdg_noalloc.cu", os.path.join(OBJ, "tdg_noalloc.o"), [])]
    for la, lb, lc, ld in QUARTET_CLASSES:
        for role in range(num_roles(la, lb, lc, ld)):   # one translation unit per (class, role): they compile in parallel
            jobs.append(("tdg_class.cu", os.path.join(OBJ, "tdg_class_%d%d%d%d_r%d.o" % (la, lb, lc, ld, role)),
                         ["-DTDG_LA=%d" % la, "-DTDG_LB=%d" % lb, "-DTDG_LC=%d" % lc, "-DTDG_LD=%d" % ld, "-DTDG_ROLE=%d" % role]
                         + CLASS_FLAGS.get((la, lb, lc, ld), [])))
    # longest compiles first (fully unrolled d-shell classes)
    jobs.sort(key=lambda j: 0 if "class" not in j[1] else -sum(int(c) for c in os.path.basename(j[1])[10:14]))
    todo = []
    for src, obj, extra in jobs:
        st = max(os.path.getmtime(os.path.join(CSRC, src)), _newest_header(src))
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < st or not _same_flags(obj, extra):
            todo.append((src, obj, extra))
    if todo:
        if verbose:
            print("compiling %d objects" % len(todo), file=sys.stderr)
        with cf.ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
            list(ex.map(_compile, todo))
    objs = [j[1] for j in jobs]
    if todo or not os.path.exists(LIB):
        cmd = [NVCC, "-shared", "-o", LIB] + objs
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("link failed:\n%s\n%s" % (r.stdout, r.stderr))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
