"""Builds the CUDA shared library in-tree: paper_1208_1186_b200/liblgf.so (sm_100a only)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "liblgf.so")
SOURCES = ["lgf_api.cu", "lgf_fft_inst.cu", "lgf_fft_inst_f64.cu", "lgf_fft_inst_f32.cu", "lgf_fft_pipe_f64.cu", "lgf_fft_pipe_f32.cu", "lgf_static.cu"]


def _headers() -> list:
    """Every header a translation unit may include: all of csrc/*.cuh plus the public C header."""
    import glob
    return sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [os.path.join(_HERE, "..", "include", "lgf.h")]


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC"]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "--cudart", "shared"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    files = [os.path.join(CSRC, f) for f in SOURCES] + _headers() + [os.path.abspath(__file__)]
    return any(os.path.getmtime(f) > t for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc-compile the library if it is missing or older than its sources (translation units in
    parallel, then one link).  Needs no GPU: nvcc cross-compiles sm_100a."""
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        objdir = os.path.join(_HERE, "build")
        os.makedirs(objdir, exist_ok=True)
        procs, objs = [], []
        for src in SOURCES:
            obj = os.path.join(objdir, src.replace(".cu", ".o"))
            objs.append(obj)
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
            procs.append((src, subprocess.Popen(cmd)))
        for src, p in procs:
            if p.wait() != 0:
                raise RuntimeError(f"nvcc failed on {src}")
        subprocess.run([nvcc] + LINK_FLAGS + ["-o", LIB + ".tmp"] + objs, check=True)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
