"""Build libf4.so (CUDA kernels + C-ABI) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libf4.so")
SOURCES = ["f4_mesh.cpp", "f4_ghost.cu", "f4_stage.cu", "f4_advect.cu", "f4_advect2.cu", "f4_fluxfix.cu", "f4_api.cu"]
HEADERS = ["f4_mesh.hpp", "f4_dev.hpp", "f4_stage_dev.cuh", os.path.join("..", "..", "include", "f4.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-cudart", "static", "-Wno-deprecated-gpu-targets"]


def _newest_source() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, f)) for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/ into the in-tree libf4.so."""
    lib = LIB
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= _newest_source():
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, os.path.splitext(src)[0] + ".o")
        objs.append(obj)
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-x", "cu", "-c", os.path.join(CSRC, src), "-o", obj]
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    for cmd, pr in procs:
        out, _ = pr.communicate()
        if verbose and out:
            print(out)
        if pr.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd) + "\n" + (out or ""))
    subprocess.check_call([nvcc, "-shared", "-cudart", "static", "-o", lib] + objs)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
