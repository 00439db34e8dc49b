"""Build liblisatdi.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2505_09600_b200.build [--force]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "liblisatdi.so")
SOURCES = [os.path.join(CSRC, "lisatdi.cu"), os.path.join(CSRC, "overlap.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("common.cuh", "dd.cuh", "orbit.cuh", "response.cuh", "fast.cuh", "chirp.cuh", "fft.cuh")] + [
    os.path.join(INCLUDE, "lisatdi.h"), os.path.join(INCLUDE, "lisatdi_bench.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "--fmad=true", "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v", "-I", INCLUDE]


def build(force=False, verbose=False):
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS)):
        return LIB
    # several ranks of one node may import the package at once: one builds (into a temporary file, renamed
    # atomically), the others wait on the lock and find the library up to date
    import fcntl
    with open(LIB + ".lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if (not force and os.path.exists(LIB)
                and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS)):
            return LIB
        tmp = f"{LIB}.{os.getpid()}.tmp"
        cmd = [NVCC, *FLAGS, "-o", tmp, *SOURCES]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            if os.path.exists(tmp):
                os.remove(tmp)
            raise RuntimeError("nvcc failed building liblisatdi.so")
        os.replace(tmp, LIB)
        if verbose:
            print(r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
