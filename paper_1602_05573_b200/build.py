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
DEPS = [CSRC / "spiir_kernels.cuh", CSRC / "spiir_layout.hpp", PKG.parent / "include" / "spiir.h"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-O3,-Wall", "-shared", "-cudart", "shared"]


PROBE_SRC = CSRC / "fp32_pipe_probe.cu"
PROBE_BIN = PKG / "fp32_pipe_probe"          # standalone microbenchmark behind the roofline ceiling in DESIGN.md section 7.1


def build_probe(force: bool = False) -> Path:
    """nvcc the FP32 pipe probe (run it on a B200: ``paper_1602_05573_b200/fp32_pipe_probe 1965``)."""
    if force or not PROBE_BIN.exists() or PROBE_SRC.stat().st_mtime > PROBE_BIN.stat().st_mtime:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = PROBE_BIN.with_suffix(f".tmp{os.getpid()}")
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                        "-o", str(tmp), str(PROBE_SRC)], check=True)
        os.replace(tmp, PROBE_BIN)
    return PROBE_BIN


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
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    print(build_probe(force="--force" in sys.argv))
