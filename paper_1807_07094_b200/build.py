"""Build libarc_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1807_07094_b200.build [--force]

The library links only the CUDA runtime; PyTorch is not involved in the build.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libarc_b200.so")
LIB_CHECKED = os.path.join(HERE, "libarc_b200_checked.so")       # -DARC_CHECKED=1: device-side bounds checks (csrc/arc_internal.cuh)

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]                 # cudart: static (nvcc default), self-contained


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "arc.h")]


def needs_build(checked: bool = False) -> bool:
    lib = LIB_CHECKED if checked else LIB
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(p) > t for p in _deps())


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: cannot build libarc_b200.so (there is no CPU fallback)")
    return p


def _compile_one(args):
    src, obj, verbose, checked = args
    cmd = [nvcc_path()] + NVCC_FLAGS + (["-DARC_CHECKED=1"] if checked else []) + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
    r = subprocess.run(cmd, capture_output=True, text=True)
    return src, r.returncode, " ".join(cmd) + "\n" + r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """Compile every csrc/*.cu to an object (in parallel: the tracer's instantiation units dominate) and link.
    checked = True: the same sources with -DARC_CHECKED=1 into libarc_b200_checked.so."""
    LIB = LIB_CHECKED if checked else globals()["LIB"]
    if not force and not needs_build(checked):
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(HERE, "build", "checked" if checked else "")
    os.makedirs(objdir, exist_ok=True)
    jobs = [(s, os.path.join(objdir, os.path.basename(s)[:-3] + ".o"), verbose, checked) for s in sources()]
    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        results = list(ex.map(_compile_one, jobs))
    for src, rc, log in results:
        if rc != 0:
            raise RuntimeError("nvcc failed:\n" + log)
        if verbose:
            sys.stderr.write(log)
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [j[1] for j in jobs]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("link failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
