"""Build libba.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension machinery)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libba.so")
SOURCES = ["ba_api.cu"]                       # unity build; the kernels are the .cuh files it includes
DEPS = ["ba_api.cu", "ba_internal.h", "ba_tables.h", "ba_enum_in.cuh", "ba_enum_out.cuh", "ba_stream.cuh", "ba_fast.cuh", "ba_peaks.cuh",
        os.path.join("..", "..", "include", "ba.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force=False, verbose=False):
    """Build (if stale) under an exclusive file lock, so that several ranks importing the binding at once (torchrun)
    do not write libba.so concurrently; the ranks that waited find it fresh."""
    import fcntl
    if not force and not needs_build():
        return LIB
    with open(os.path.join(HERE, ".build.lock"), "w") as lk:
        fcntl.flock(lk, fcntl.LOCK_EX)
        try:
            if not force and not needs_build():
                return LIB
            return _build(verbose)
        finally:
            fcntl.flock(lk, fcntl.LOCK_UN)


def _build(verbose):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + \
          [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
