"""In-tree native builds (no JIT cache: the built .so files travel with the repo snapshot).

    libibp.so          csrc/*.cu + csrc/*.cpp, nvcc, sm_100a only   -> the C-ABI product library (include/ibp.h)
    libibp_datagen.so  datagen/ibp_datagen.c, gcc                   -> seeded input generators

A target is rebuilt when any of its sources (or headers) is newer than the .so.
"""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
LIB = PKG / "libibp.so"
DATAGEN_LIB = PKG / "datagen" / "libibp_datagen.so"

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC,-O3,-fopenmp,-mbmi2,-mpopcnt,-Wall",
    "-shared", "-cudart", "static",
]


def _stale(target: Path, sources) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(Path(s).stat().st_mtime > t for s in sources)


def _run(cmd, verbose):
    if verbose:
        print("+", " ".join(str(c) for c in cmd), flush=True)
    r = subprocess.run([str(c) for c in cmd], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"build failed: {' '.join(str(c) for c in cmd)}\n{r.stdout}\n{r.stderr}")
    if verbose and (r.stdout or r.stderr):
        print(r.stdout, r.stderr, flush=True)


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: the IBP library is CUDA-only (sm_100a) and has no CPU fallback")
    return p


def build_library(force: bool = False, verbose: bool = False, extra_flags=()) -> Path:
    src = sorted((PKG / "csrc").glob("*.cu")) + sorted((PKG / "csrc").glob("*.cpp"))
    deps = src + sorted((PKG / "csrc").glob("*.h")) + sorted((PKG / "csrc").glob("*.cuh")) + sorted((ROOT / "include").glob("*.h"))
    if force or _stale(LIB, deps):
        tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")       # per process: concurrent builds (torchrun ranks, test workers) do not collide
        _run([nvcc_path(), *NVCC_FLAGS, *extra_flags, "-I", ROOT / "include", "-I", PKG / "csrc", "-x", "cu", *src,
              "-o", tmp, "-lgomp", "-lrt"], verbose)
        os.replace(tmp, LIB)
    return LIB


def build_datagen(force: bool = False, verbose: bool = False) -> Path:
    src = PKG / "datagen" / "ibp_datagen.c"
    if force or _stale(DATAGEN_LIB, [src]):
        tmp = DATAGEN_LIB.with_suffix(f".so.tmp{os.getpid()}")
        _run(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", src, "-o", tmp, "-lm"], verbose)
        os.replace(tmp, DATAGEN_LIB)
    return DATAGEN_LIB


def build_all(force: bool = False, verbose: bool = False):
    return build_library(force, verbose), build_datagen(force, verbose)


if __name__ == "__main__":
    build_all(force=True, verbose=True)
