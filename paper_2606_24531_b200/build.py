"""Build step: compile the CUDA path into the in-tree C-ABI library ``libaceapex.so`` (sm_100a only).

``python -m paper_2606_24531_b200.build`` or ``build()``; nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_DIR, "csrc")
SO = os.path.join(_DIR, "libaceapex.so")
SOURCES = ["aceapex.cu"]
HEADERS = ["format.cuh", "entropy.cuh", "match.cuh", "seek.cuh"]
INCLUDE = os.path.join(os.path.dirname(_DIR), "include", "aceapex.h")

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")
    return exe


def stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [INCLUDE]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return SO
    tmp = SO + f".tmp{os.getpid()}"
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed")
    if verbose:
        sys.stderr.write(r.stdout + r.stderr)
    os.replace(tmp, SO)
    return SO


def build_variant(name: str, defines: dict, verbose: bool = False) -> str:
    """Compile the library with extra -D macros (the granularity knobs of PAPER.md:86-92 in this design:
    ACEAPEX_MATCH_THREADS, ACEAPEX_ENTROPY_WARPS) into build/libaceapex_<name>.so; `bench.py --sweep` loads
    such a variant through the ACEAPEX_LIB environment variable."""
    out_dir = os.path.join(_DIR, "build")
    os.makedirs(out_dir, exist_ok=True)
    so = os.path.join(out_dir, f"libaceapex_{name}.so")
    flags = [f"-D{k}={v}" for k, v in sorted(defines.items())]
    cmd = [nvcc()] + NVCC_FLAGS + flags + (["-Xptxas", "-v"] if verbose else []) + ["-o", so] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed")
    return so


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
