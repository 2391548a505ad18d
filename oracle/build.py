"""Build the CPU oracle (TEST INFRASTRUCTURE) with gcc.  No CUDA, no torch.

    python -m oracle.build

-O2 only: no -ffast-math, so the fp64 sums keep the order written in xengine_oracle.c.
"""
import fcntl
import os
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "xengine_oracle.c")
LIB = os.path.join(HERE, "libxoracle.so")
CFLAGS = ["-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]


def _stale():
    return not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC)


def build(force: bool = False) -> str:
    """Compile the oracle if missing or stale; concurrent callers serialise on a file lock (see the product's build.py)."""
    if not force and not _stale():
        return LIB
    with open(LIB + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not _stale():
                return LIB
            fd, tmp = tempfile.mkstemp(prefix="libxoracle.", suffix=".so.tmp", dir=HERE)
            os.close(fd)
            cmd = ["gcc"] + CFLAGS + [SRC, "-o", tmp, "-lm"]
            subprocess.run(cmd, check=True)
            os.chmod(tmp, 0o755)
            os.replace(tmp, LIB)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
