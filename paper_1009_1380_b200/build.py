"""Build libradon_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libradon_b200.so")
SOURCES = ["api.cu", "gridding.cu", "fft2d.cu", "fft2d_composite.cu", "proj.cu", "filter.cu", "paper_bins.cu", "plan_device.cu", "plan_host.cpp"]
HEADERS = ["kernels.h", "radon_internal.h", "fft_device.cuh", "async_copy.cuh", "taps.cuh", "plan_device.h", os.path.join("..", "..", "include", "radon.h")]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-shared", "-Xcompiler", "-fPIC",
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-lpthread",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    flags = [f for f in NVCC_FLAGS if f not in ("-shared", "-lpthread")] + (["-Xptxas", "-v"] if verbose else [])
    flags += os.environ.get("RADON_NVCC_DEFS", "").split()      # tuning builds: -DRADON_...=...
    # one nvcc per translation unit, side by side (the FFT templates dominate the build time)
    procs, objs = [], []
    for f in SOURCES:
        obj = os.path.join(objdir, os.path.splitext(f)[0] + ".o")
        objs.append(obj)
        procs.append(subprocess.Popen([nvcc] + flags + ["-c", os.path.join(CSRC, f), "-o", obj]))
    failed = [f for f, pr in zip(SOURCES, procs) if pr.wait() != 0]
    if failed:
        raise subprocess.CalledProcessError(1, "nvcc -c " + " ".join(failed))
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs + ["-lpthread"], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
