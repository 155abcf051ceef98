"""Build the CUDA library (libradt.so) in-tree for sm_100a with nvcc.  No JIT cache, no torch types.

Every source is compiled to its own object (in parallel, only when it or a header changed) and the objects are linked into
libradt.so; the ptxas resource report of all kernels goes to build_ptxas.log."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libradt.so")
SOURCES = ["radt_api.cu", "radt_setup.cu", "radt_march.cu", "radt_march_win.cu", "radt_microbench.cu", "radt_disk.cu", "radt_mlp_tc.cu", "radt_mlp_tc_bwd.cu"]
HEADERS = ["radt_dev.cuh", "radt_kernels.h", "radt_march.cuh", "radt_tc.cuh", os.path.join("..", "..", "include", "radt.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _compile(nvcc, src, obj):
    cmd = [nvcc] + NVCC_FLAGS + ["-c", "-o", obj, os.path.join(CSRC, src)]
    res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
    return src, cmd, res


def build(force: bool = False, verbose: bool = False) -> str:
    hdr_time = max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)
    hdr_time = max(hdr_time, os.path.getmtime(os.path.abspath(__file__)))
    os.makedirs(OBJ, exist_ok=True)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    todo = []
    for s in SOURCES:
        o = os.path.join(OBJ, s[:-3] + ".o")
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(hdr_time, os.path.getmtime(os.path.join(CSRC, s))):
            todo.append((s, o))
    objs = [os.path.join(OBJ, s[:-3] + ".o") for s in SOURCES]
    if not todo and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(o) for o in objs):
        return LIB
    with ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as ex:
        results = list(ex.map(lambda so: _compile(nvcc, *so), todo))
    logs = []
    for src, cmd, res in results:
        if verbose or res.returncode != 0:
            print(res.stdout)
            print(res.stderr)
        if res.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}")
        with open(os.path.join(OBJ, src[:-3] + ".ptxas.log"), "w") as f:
            f.write(" ".join(cmd) + "\n" + res.stderr)
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs
    res = subprocess.run(link, cwd=CSRC, capture_output=True, text=True)
    if res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
        raise RuntimeError("nvcc link failed")
    for s in SOURCES:
        p = os.path.join(OBJ, s[:-3] + ".ptxas.log")
        if os.path.exists(p):
            with open(p) as f:
                logs.append(f.read())
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        f.write("\n".join(logs))
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=False))
