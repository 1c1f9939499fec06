"""Builds libsn_poisson.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

The kernels of every box shape live in their own translation unit (csrc/shape_tu.cu compiled once per -DSNP_TU=<n>,
see csrc/shapes.cuh), so the objects are compiled in parallel and linked into one shared library."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsn_poisson.so")
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-fmad=false",                              # pinned fp64 expression trees (R10)
    "-Xcompiler", "-fPIC,-ffp-contract=off,-O2",
]
SHAPE_TUS = list(range(11)) + [100, 200]        # csrc/shapes.cuh: kNumResShapes resident shapes, blocked, dispatch


def units():
    """(source, object, extra flags) of every translation unit."""
    out = [(os.path.join(CSRC, f), os.path.join(OBJ, f[:-3] + ".o"), [])
           for f in sorted(os.listdir(CSRC)) if f.endswith(".cu") and f != "shape_tu.cu"]
    out += [(os.path.join(CSRC, "shape_tu.cu"), os.path.join(OBJ, f"shape_tu_{n}.o"), [f"-DSNP_TU={n}"])
            for n in SHAPE_TUS]
    return out


def _deps():
    return [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [
        os.path.join(os.path.dirname(HERE), "include", f) for f in ("sn_poisson.h", "sn_levelset.h", "sn_weno.h")]


def _stale(target: str) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in _deps())


def build(force: bool = False, verbose: bool = False, only=None, extra_flags=()) -> str:
    """`only`: iterable of SNP_TU numbers to recompile (development shortcut; everything else must be up to date).
    `extra_flags`: additional nvcc flags (A/B builds such as -DSNP_GROUP_ROWS_ROOMY=2).  Only the command line below
    passes any -- from SN_NVCC_EXTRA --; the library callers (`__graft_entry__.build()`, the tests) never do, so the
    environment cannot change what they build."""
    if not force and only is None and not extra_flags and not _stale(LIB):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    todo = []
    for src, obj, extra in units():
        if only is not None:
            tu = extra[0].split("=")[1] if extra else os.path.basename(src)
            if str(tu) not in {str(o) for o in only} and os.path.exists(obj):
                continue
        elif not force and not _stale(obj):
            continue
        todo.append([nvcc, *NVCC_FLAGS, *extra_flags, *(["-Xptxas", "-v"] if verbose else []), *extra, "-c", src, "-o", obj])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(" ".join(cmd[-4:]) + "\n" + r.stdout + r.stderr)
        if r.returncode:
            raise subprocess.CalledProcessError(r.returncode, cmd)

    with ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as ex:
        list(ex.map(run, todo))
    subprocess.check_call([nvcc, "-shared", "-o", LIB, *[obj for _, obj, _ in units()]])
    return LIB


if __name__ == "__main__":
    only = [a.split("=")[1].split(",") for a in sys.argv if a.startswith("--only=")]
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, only=only[0] if only else None,
                extra_flags=tuple(os.environ.get("SN_NVCC_EXTRA", "").split())))
