"""Build the CUDA library (libradt.so) in-tree for sm_100a with nvcc.  No JIT cache, no torch types."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libradt.so")
SOURCES = ["radt_api.cu", "radt_setup.cu", "radt_march.cu", "radt_march_win.cu", "radt_microbench.cu", "radt_disk.cu", "radt_mlp.cu", "radt_mlp_tc.cu"]
HEADERS = ["radt_dev.cuh", "radt_kernels.h", "radt_march.cuh", os.path.join("..", "..", "include", "radt.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def build(force: bool = False, verbose: bool = False) -> str:
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed")
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=False))
