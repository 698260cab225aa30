"""Build librosen.so (C ABI + sm_100a kernels) in-tree with nvcc.

    python -m paper_1704_04381_b200.build [--force]

nvcc cross-compiles for sm_100a without a GPU. The library is linked against the static CUDA
runtime so that it loads wherever a driver is present (and still dlopen()s on a CPU-only box,
where every generate call then fails loudly with ROSEN_ECUDA -- there is no CPU fallback).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["api.cu", "lattice.cu", "lattice_hash.cu", "lattice_model.cu", "lattice_perm.cu", "realspace.cu", "realspace_long.cu", "reduce.cu"]
HEADERS = ["common.cuh", "direction.cuh", "philox.cuh", "reduce.cuh", os.path.join("..", "..", "include", "rosen.h")]
TARGET = os.path.join(HERE, "librosen.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]
    if not force and os.path.exists(TARGET) and all(os.path.getmtime(TARGET) >= os.path.getmtime(d) for d in deps):
        return TARGET
    objs = []
    procs = []
    for s in srcs:
        o = s[:-3] + ".o"
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", s, "-o", o]
        procs.append((cmd, subprocess.Popen(cmd)))
        objs.append(o)
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    link = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static",
            "-Xcompiler", "-fPIC", "-o", TARGET] + objs
    subprocess.run(link, check=True)
    return TARGET


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
