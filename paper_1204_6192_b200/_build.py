"""In-tree build of the C-ABI library ``lib/libhsg.so`` (CUDA, sm_100a only).

``nvcc`` cross-compiles without a GPU (one translation unit per lattice size of the sweep kernel, compiled in parallel), so this runs on the CPU box (``__graft_entry__.build()``) and on
the GPU box alike.  The shared object is rebuilt when any source under ``csrc/`` or ``include/hsg.h``
is newer than it.
"""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

_PKG = Path(__file__).resolve().parent
_ROOT = _PKG.parent
CSRC = _PKG / "csrc"
HEADER = _ROOT / "include" / "hsg.h"
LIB = _PKG / "lib" / "libhsg.so"

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-fmad=false",            # no compiler-chosen multiply-add fusion; every FMA is explicit
    "-Xcompiler", "-fPIC",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the hsg CUDA library cannot be built (there is no CPU fallback)")


def sources():
    return sorted(CSRC.glob("*.cu")) + sorted(CSRC.glob("*.cuh")) + [HEADER]


def stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in sources())


def build(force: bool = False, verbose: bool = False) -> Path:
    """Compile every translation unit under csrc/ (in parallel) and link lib/libhsg.so; returns its path."""
    if not force and not stale():
        return LIB
    LIB.parent.mkdir(parents=True, exist_ok=True)
    objdir = LIB.parent / f"obj.tmp{os.getpid()}"
    objdir.mkdir(parents=True, exist_ok=True)
    nvcc = _nvcc()
    units = sorted(CSRC.glob("*.cu"))
    cmds = [[nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", str(u), "-o", str(objdir / (u.stem + ".o"))] for u in units]
    try:
        procs = [subprocess.Popen(c, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True) for c in cmds]
        outs = [p.communicate()[0] for p in procs]
        for c, p, o in zip(cmds, procs, outs):
            if p.returncode != 0:
                raise RuntimeError("nvcc failed:\n" + " ".join(c) + "\n" + o)
            if verbose:
                print(o)
        tmp = LIB.with_name(f"libhsg.tmp{os.getpid()}.so")
        link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC",
                *[str(objdir / (u.stem + ".o")) for u in units], "-o", str(tmp)]
        res = subprocess.run(link, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("link failed:\n" + " ".join(link) + "\n" + res.stdout + res.stderr)
        os.replace(tmp, LIB)
    finally:
        shutil.rmtree(objdir, ignore_errors=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
