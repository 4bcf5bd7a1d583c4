"""Builds the C-ABI shared library in-tree with nvcc for sm_100a.

    python -m paper_1909_05423_b200.build [--force]

The .so is git-ignored (history stays source-only) but travels with the working tree.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG_DIR, "csrc")
INCLUDE = os.path.join(os.path.dirname(PKG_DIR), "include")
LIB_PATH = os.path.join(PKG_DIR, "libpittpack_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]
OBJ_DIR = os.path.join(PKG_DIR, "build")          # git-ignored


def sources():
    out = [os.path.join(INCLUDE, "pittpack_b200.h")]
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, name))
    return out


def is_stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(s) > t for s in sources())


def find_nvcc() -> str:
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        raise RuntimeError("nvcc not found: cannot build libpittpack_b200.so")
    return nvcc


def translation_units():
    return sorted(n for n in os.listdir(CSRC) if n.endswith(".cu"))


def build(force: bool = False, verbose: bool = False, defines=(), out: str = LIB_PATH) -> str:
    """Compile every csrc/*.cu for sm_100a (in parallel: one nvcc per translation unit) and link them into
    the shared library.  `defines`: extra -D flags (tuning switches of the kernels); `out`: library path."""
    if not force and not defines and out == LIB_PATH and not is_stale():
        return LIB_PATH
    from concurrent.futures import ThreadPoolExecutor
    nvcc = find_nvcc()
    obj_dir = OBJ_DIR if out == LIB_PATH else out + ".obj"
    os.makedirs(obj_dir, exist_ok=True)

    def compile_one(name):
        obj = os.path.join(obj_dir, name[:-3] + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *defines, "-c", "-o", obj, os.path.join(CSRC, name)]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        res = subprocess.run(cmd, capture_output=True, text=True)
        return name, obj, res

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as pool:
        results = list(pool.map(compile_one, translation_units()))
    for name, _, res in results:
        if res.returncode != 0:
            raise RuntimeError(f"nvcc failed on {name}:\n" + res.stdout + res.stderr)
        if verbose:
            print(f"==== {name}\n{res.stderr}")
    cmd = [nvcc, *LINK_FLAGS, "-o", out, *[obj for _, obj, _ in results]]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + res.stdout + res.stderr)
    return out


if __name__ == "__main__":
    # python -m paper_1909_05423_b200.build [--force] [-v] [-DNAME=VALUE ...] [-o other.so]
    out_path = sys.argv[sys.argv.index("-o") + 1] if "-o" in sys.argv else LIB_PATH
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv,
                defines=tuple(a for a in sys.argv[1:] if a.startswith("-D")), out=out_path))
