"""Build the C-ABI CUDA library ``libmphv.so`` in-tree with nvcc for sm_100a.

Usage: ``python -m paper_2305_01487_b200.build [--force]``. nvcc cross-compiles without
a GPU; the built .so is git-ignored but travels to the GPU box with the snapshot.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
SO = PKG / "libmphv.so"
SOURCES = [CSRC / "mphv.cu", CSRC / "mphv_coupled.cu", CSRC / "mphv_noalloc.cu"]
DEPS = SOURCES + sorted(CSRC.glob("*.cuh")) + [ROOT / "include" / "mphv.h"]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found (set NVCC=/path/to/nvcc)")


def up_to_date() -> bool:
    return SO.exists() and all(SO.stat().st_mtime >= p.stat().st_mtime for p in DEPS)


def build(force: bool = False, verbose: bool = False, extra: list[str] | None = None) -> Path:
    if not force and up_to_date():
        return SO
    tmp = SO.with_suffix(f".{os.getpid()}.tmp")
    objs = [PKG / f".{src.stem}.{os.getpid()}.o" for src in SOURCES]
    cmds = [[nvcc(), *NVCC_FLAGS, *(extra or []), *(["-Xptxas", "-v"] if verbose else []),
             "-I", str(ROOT / "include"), "-c", "-o", str(o), str(src)] for src, o in zip(SOURCES, objs)]
    procs = [subprocess.Popen(c, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for c in cmds]   # in parallel
    outs = [p.communicate() for p in procs]
    try:
        for c, p, (so, se) in zip(cmds, procs, outs):
            if verbose:
                sys.stderr.write(se)
            if p.returncode != 0:
                raise RuntimeError("nvcc failed:\n" + " ".join(c) + "\n" + so + se)
        link = [nvcc(), *LINK_FLAGS, "-o", str(tmp), *map(str, objs)]
        r = subprocess.run(link, capture_output=True, text=True)
        if r.returncode != 0:
            tmp.unlink(missing_ok=True)
            raise RuntimeError("nvcc link failed:\n" + " ".join(link) + "\n" + r.stdout + r.stderr)
    finally:
        for o in objs:
            o.unlink(missing_ok=True)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
