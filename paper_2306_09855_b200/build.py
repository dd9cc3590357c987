"""Build step: compile the CUDA sources under csrc/ into the in-tree shared library libnc.so
(sm_100a only, -lineinfo so that ncu's source page maps to the .cu/.cuh files)."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libnc.so"
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

NVCC_FLAGS = [
    "-O3", "-std=c++17",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-Xptxas", "-v",
    "-cudart", "static",
]


def sources():
    return sorted(CSRC.glob("*.cu")), (sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.inl")) + sorted(CSRC.glob("*.h")) +
                                     sorted((HERE.parent / "include").glob("*.h")))


def build(force: bool = False, verbose: bool = False) -> Path:
    cus, deps = sources()
    if not force and LIB.exists():
        newest = max(p.stat().st_mtime for p in cus + deps)
        if LIB.stat().st_mtime >= newest:
            return LIB
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [NVCC, *NVCC_FLAGS, *os.environ.get("NC_NVCC_EXTRA", "").split(), "-o", str(tmp), *map(str, cus)]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libnc.so")
    (HERE / "ptxas_info.txt").write_text(r.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
    print(LIB)
