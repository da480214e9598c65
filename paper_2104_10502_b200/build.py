"""Build libqe_hpsi.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot).

    python -m paper_2104_10502_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libqe_hpsi.so")
SOURCES = ["qe_hpsi.cu"]
HEADERS = ["fft_core.cuh", "fft_kernels.cuh", "fft2p_kernels.cuh", "fft3p_kernels.cuh", "fft2t_kernels.cuh", "zgemm_kernels.cuh", "zgemm_tma_kernels.cuh", "ozaki_kernels.cuh", "cert_kernels.cuh",
           os.path.join("..", "..", "include", "qe_hpsi.h"), os.path.join("..", "..", "include", "qe_hpsi_test.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC,-ffp-contract=off",
    "-shared",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the CUDA library if it is missing or older than its sources. Returns the path of the .so."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + \
        [os.path.join(CSRC, s) for s in SOURCES]
    proc = subprocess.run(cmd, capture_output=True, text=True)
    if proc.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + proc.stdout + proc.stderr)
    if verbose:
        sys.stderr.write(proc.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
