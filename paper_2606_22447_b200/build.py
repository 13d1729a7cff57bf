"""Build libvcsb200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
SO = os.path.join(PKG, "libvcsb200.so")
SOURCES = ["vcs_api.cu", "vcs_step.cu", "vcs_peak.cu"]
HEADERS = ["vcs_decode.cuh", "vcs_tia.cuh", "vcs_state.cuh", "vcs_step.cuh", "vcs_optable.cuh", os.path.join("..", "..", "include", "vcs.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--use_fast_math",
              "-maxrregcount=56"]     # caps the out-of-line device functions (the kernels carry __launch_bounds__): round 1 measured 9.70 -> 9.51 ms
                                      # on config 4 with 48; on the round-2 kernel 40 / 48 / 56 / 64 / 80 give 7.05 / 6.97 / 6.92 / 7.15 / 7.10 ms


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = SO + f".tmp{os.getpid()}"
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, f) for f in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libvcsb200.so")
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force=True, verbose=True))
