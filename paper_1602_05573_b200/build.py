"""Build the C-ABI shared library libspiir_b200.so in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libspiir_b200.so"
SOURCES = [CSRC / "spiir_api.cu"]
DEPS = [CSRC / "spiir_kernels.cuh", CSRC / "spiir_layout.hpp", PKG.parent / "include" / "spiir.h", PKG / "sass_tune.py"]
# -no-compress: the SASS post-pass (sass_tune.py) patches the kernels' bytes inside the finished library
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-O3,-Wall", "-shared", "-cudart", "shared", "-no-compress"]


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in SOURCES + DEPS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", str(tmp), *map(str, SOURCES)]
        subprocess.run(cmd, check=True)
        if os.environ.get("SPIIR_NO_SASS_TUNE") != "1":
            # operand-reuse triples in the tile bodies (sass_tune.py: verified block by block, bitwise-neutral); a library the
            # pass cannot read is shipped as ptxas wrote it
            try:
                from . import sass_tune
            except ImportError:
                import sass_tune
            try:
                stats = sass_tune.tune_library(tmp)
                if verbose:
                    print("sass_tune:", stats)
            except Exception as e:      # noqa: BLE001
                print(f"sass_tune skipped: {e!r}", file=sys.stderr)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
