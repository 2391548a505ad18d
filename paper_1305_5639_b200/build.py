"""Build libcorr.so (the C-ABI X-engine library) in-tree with nvcc for sm_100a.

    python -m paper_1305_5639_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The CUDA runtime is linked statically, so the library has
no dependency on torch (callers pass plain device pointers and a cudaStream_t).
"""
import fcntl
import os
import subprocess
import sys
import tempfile

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


def _stale():
    if not os.path.exists(LIB):
        return True
    newest = max(os.path.getmtime(d) for d in _deps() + [os.path.abspath(__file__)])
    return os.path.getmtime(LIB) < newest


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libcorr.so if it is missing or older than its sources.  Safe when several processes (torchrun ranks)
    call it at once: one compiles under a file lock into its own temporary file, the others wait and find it built."""
    if not force and not _stale():
        return LIB
    with open(LIB + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not _stale():          # another process built it while this one waited for the lock
                return LIB
            fd, tmp = tempfile.mkstemp(prefix="libcorr.", suffix=".so.tmp", dir=HERE)
            os.close(fd)
            cmd = [_nvcc()] + NVCC_FLAGS + ["-I", INCLUDE]
            # developer A/B builds, e.g. CORR_EXTRA_NVCC_FLAGS=-DCORR_FEED_RELEASE_ARRIVE (csrc/ptx.cuh); always with --force
            cmd += os.environ.get("CORR_EXTRA_NVCC_FLAGS", "").split()
            if verbose:
                cmd += ["-Xptxas", "-v"]
            cmd += _sources() + ["-o", tmp]
            res = subprocess.run(cmd, capture_output=True, text=True)
            if res.returncode != 0:
                sys.stderr.write(res.stdout + res.stderr)
                if os.path.exists(tmp):
                    os.unlink(tmp)
                raise RuntimeError("nvcc failed building libcorr.so")
            if verbose:
                sys.stderr.write(res.stdout + res.stderr)
            os.chmod(tmp, 0o755)
            os.replace(tmp, LIB)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
