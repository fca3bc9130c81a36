"""Build libbt.so (the C-ABI library, include/bt.h) in-tree with nvcc for sm_100a.

    python -m paper_2208_02382_b200._build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libbt.so")
SOURCES = ["bt_api.cu", "track.cu", "grid.cu", "sort.cu", "moments.cu", "poisson.cu", "calib.cu"]
HEADERS = [os.path.join(CSRC, "bt_internal.h"), os.path.join(CSRC, "grid_dev.cuh"), os.path.join(CSRC, "bulk_copy.cuh"), os.path.join(HERE, "..", "include", "bt.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",            # FMA contraction allowed on the GPU side (R14); canonical CIC weights use _rn intrinsics
    "-Xcompiler", "-fPIC,-O2,-Wall",
    "-shared", "-cudart", "shared",
]


# cuFFT (the FFT of the Poisson solve is a library step); rpath so that the image's CUDA 12.9 copy is found at load time
LINK = ["-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    return "nvcc"


STAMP = LIB + ".stamp"


def _digest():
    """Content hash of sources + flags (mtimes do not survive the trip to the GPU box)."""
    import hashlib
    h = hashlib.sha256(" ".join(NVCC_FLAGS + LINK).encode())
    for d in [os.path.join(CSRC, s) for s in SOURCES] + HEADERS:
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def needs_build():
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as f:
        return f.read().strip() != _digest()


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES] + LINK
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    with open(STAMP, "w") as f:
        f.write(_digest())
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
