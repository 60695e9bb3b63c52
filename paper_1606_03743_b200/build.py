"""Builds libbemcub.so (the C-ABI CUDA library, include/bemcub.h) in-tree with nvcc for sm_100a.

    python -m paper_1606_03743_b200.build [--force]

nvcc cross-compiles without a GPU; the .so is git-ignored but travels with the working tree.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
# BEMCUB_LIB: load another build of the same library (A/B timing of kernel variants); never rebuilt, so it
# may not match csrc/ - the binding says so on stderr when it loads it, and the tests and bench.py refuse it
# unless BEMCUB_LIB_ALLOW=1 is set as well (override_active / override_refused below)
LIB = Path(os.environ["BEMCUB_LIB"]) if os.environ.get("BEMCUB_LIB") else PKG / "libbemcub.so"
SOURCES = [CSRC / "bemcub.cu"]
DEPS = sorted(CSRC.glob("*.cu*")) + sorted(CSRC.glob("*.h")) + sorted(CSRC.glob("*.inl")) + [PKG.parent / "include" / "bemcub.h"]

NVCC_FLAGS = [
    "-shared", "-Xcompiler", "-fPIC", "-O3", "-std=c++17",
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
]


def override_active() -> bool:
    return bool(os.environ.get("BEMCUB_LIB"))


def override_refused() -> bool:
    """True where results must describe the sources in this tree (tests, bench.py) and BEMCUB_LIB points elsewhere."""
    return override_active() and os.environ.get("BEMCUB_LIB_ALLOW") != "1"


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the bemcub CUDA library cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if os.environ.get("BEMCUB_LIB"):
        return False
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(d.stat().st_mtime > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not is_stale():
        return LIB
    cmd = [nvcc_path(), *NVCC_FLAGS, "-o", str(LIB), *map(str, SOURCES)]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
