"""Build librbg.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2308_04869_b200.build [--force]

-fmad=false and -ffp-contract=off: no implicit FMA contraction on device or host; the kernels
spell every fused operation as fma().  -lineinfo keeps ncu's source page usable.
No -split-compile: with it the generated code of the sample loop differed from build to build on this machine (505 or
618 instructions for the same source, a 12 % difference in throughput); a single ptxas pass is reproducible.
"""
from __future__ import annotations

import hashlib
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
SOURCES = [PKG / "csrc" / "rbg.cu"]
DEPS = SOURCES + [PKG / "csrc" / "rbg_kernels.cuh", PKG / "csrc" / "rbg_be_kernels.cuh", ROOT / "include" / "rbg.h"]
LIB = PKG / "librbg.so"
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-O2", "-shared", "--ptxas-options=-v"]


def _digest() -> str:
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for p in DEPS:
        h.update(p.read_bytes())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> Path:
    """checked = True builds librbg_checked.so with -DRBG_CHECKED (device-side index / layout / ring-slot checks, include/rbg.h
    rbg_selfcheck_failures) next to the normal library."""
    lib = PKG / "librbg_checked.so" if checked else LIB
    tag = PKG / (".librbg_checked.tag" if checked else ".librbg.tag")
    dig = _digest()
    if not force and lib.exists() and tag.exists() and tag.read_text() == dig:
        return lib
    cmd = ["nvcc", *NVCC_FLAGS, *(["-DRBG_CHECKED"] if checked else []), "-o", str(lib), *map(str, SOURCES)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if not checked:
        (PKG / "ptxas.log").write_text(res.stderr)
    if res.returncode != 0:
        sys.stderr.write(res.stderr)
        raise RuntimeError("nvcc failed building librbg.so")
    if verbose:
        sys.stderr.write(res.stderr)
    tag.write_text(dig)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True, checked="--checked" in sys.argv))
