"""Build libcorr.so (the C-ABI X-engine library) in-tree with nvcc for sm_100a.

    python -m paper_1305_5639_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The CUDA runtime is linked statically, so the library has
no dependency on torch (callers pass plain device pointers and a cudaStream_t).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libcorr.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-cudart", "static",
]


def _sources():
    return [os.path.join(CSRC, "corr.cu")]


def _deps():
    deps = [os.path.join(INCLUDE, "corr.h")]
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh", ".h")):
            deps.append(os.path.join(CSRC, f))
    return deps


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(d) for d in _deps() + [os.path.abspath(__file__)])
        if os.path.getmtime(LIB) >= newest:
            return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + ["-I", INCLUDE]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    if os.environ.get("CORR_DEFINES"):        # developer build: extra -D switches for A/B experiments
        cmd += os.environ["CORR_DEFINES"].split()
    if os.environ.get("CORR_STATS"):          # developer build: per-role stall counters (clock64) in the pair kernel
        cmd += ["-DCORR_STATS"]
    cmd += _sources() + ["-o", LIB + ".tmp"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libcorr.so")
    if verbose:
        sys.stderr.write(res.stdout + res.stderr)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
