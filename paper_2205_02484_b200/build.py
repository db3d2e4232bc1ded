"""Build paper_2205_02484_b200/libcuharm.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2205_02484_b200.build [--force] [--verbose]

The library links the CUDA runtime statically and has no other dependency (no torch, no Python).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INC = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libcuharm.so")
SOURCES = ["cuharm_api.cu", "cuharm_noalloc.cu"]
DEPS = ["cuharm_api.cu", "cuharm_noalloc.cu", "cuharm_phys.cuh", "cuharm_geom.cuh", "cuharm_flux.cuh", "cuharm_kernels.cuh", "cuharm_chain.cuh",
        "cuharm_update_tmap.cuh"]


def nvcc_path() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in DEPS] + [os.path.join(INC, "cuharm.h")]
    return any(os.path.getmtime(f) > t for f in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "--shared", "-Xcompiler", "-fPIC,-O2,-Wall", "-cudart", "static", "-I", INC, "-o", LIB]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
