"""In-tree build of the C-ABI library ``lib/libhsg.so`` (CUDA, sm_100a only).

``nvcc`` cross-compiles without a GPU (one translation unit per lattice size of the sweep kernel, compiled in parallel), so this runs on the CPU box (``__graft_entry__.build()``) and on
the GPU box alike.  The shared object is rebuilt when the contents of any source under ``csrc/`` or of
``include/hsg.h`` (or the compiler flags) differ from what it was built from: a digest kept beside it, not file
times, so that a copy of the tree whose times were not preserved is not rebuilt.
"""
from __future__ import annotations

import hashlib
import os
import re
import shutil
import subprocess
from pathlib import Path

_PKG = Path(__file__).resolve().parent
_ROOT = _PKG.parent
CSRC = _PKG / "csrc"
HEADER = _ROOT / "include" / "hsg.h"
LIB = _PKG / "lib" / "libhsg.so"
DIGEST = _PKG / "lib" / "libhsg.sources.sha256"

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
    return sorted(CSRC.glob("*.cu")) + sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.h")) + [HEADER]


def _digest() -> str:
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for p in sources():
        h.update(p.name.encode()); h.update(b"\0"); h.update(p.read_bytes()); h.update(b"\0")
    return h.hexdigest()


def stale() -> bool:
    if not LIB.exists() or not DIGEST.exists():
        return True
    return DIGEST.read_text().strip() != _digest()


def _deps(unit: Path) -> set:
    """The files a translation unit includes (quoted includes, transitively)."""
    seen, todo = set(), [unit]
    while todo:
        f = todo.pop()
        if f in seen or not f.exists():
            continue
        seen.add(f)
        for m in re.finditer(r'#include\s+"([^"]+)"', f.read_text()):
            todo.append((f.parent / m.group(1)).resolve())
    return seen


def _unit_digest(unit: Path) -> str:
    """Digest of a translation unit: the compiler flags and the contents of every file it includes."""
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for p in sorted(_deps(unit)):
        h.update(p.name.encode()); h.update(b"\0"); h.update(p.read_bytes()); h.update(b"\0")
    return h.hexdigest()


def _unit_digest_file(obj: Path) -> Path:
    return obj.with_suffix(".sha256")


def build(force: bool = False, verbose: bool = False) -> Path:
    """Compile the translation units under csrc/ whose sources changed (in parallel; objects are kept under lib/obj/) and
    link lib/libhsg.so; returns its path.  Fails loudly: there is no CPU fallback."""
    if not force and not stale():
        return LIB
    objdir = LIB.parent / "obj"
    objdir.mkdir(parents=True, exist_ok=True)
    nvcc = _nvcc()
    units = sorted(CSRC.glob("*.cu"))
    todo = []
    for u in units:
        o = objdir / (u.stem + ".o")
        d = _unit_digest_file(o)
        if force or not o.exists() or not d.exists() or d.read_text().strip() != _unit_digest(u):
            todo.append((u, o))
    cmds = [[nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", str(u), "-o", str(o)] for u, o in todo]
    procs = [subprocess.Popen(c, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True) for c in cmds]
    outs = [p.communicate()[0] for p in procs]
    for c, p, o in zip(cmds, procs, outs):
        if p.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + " ".join(c) + "\n" + o)
        if verbose:
            print(o)
    for u, o in todo:
        _unit_digest_file(o).write_text(_unit_digest(u))
    tmp = LIB.with_name(f"libhsg.tmp{os.getpid()}.so")
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC",
            *[str(objdir / (u.stem + ".o")) for u in units], "-o", str(tmp)]
    res = subprocess.run(link, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + " ".join(link) + "\n" + res.stdout + res.stderr)
    os.replace(tmp, LIB)
    DIGEST.write_text(_digest())
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
