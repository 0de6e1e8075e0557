"""Build the C-ABI CUDA library (csrc/*.cu -> libspinllg.so, in-tree) for sm_100a with nvcc.

Usage: python -m paper_1901_11350_b200.build [--force] [--verbose]
nvcc cross-compiles without a GPU; the resulting .so travels to the GPU box with the repo snapshot.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libspinllg.so")
SOURCES = ["spin_api.cu", "spin_ddi.cu", "spin_jit.cu"]
HEADERS = ["spinllg_internal.h", "spin_kernels.cuh", "spin_device_math.cuh", "spin_jit_kernels.cuh", "spin_jit_march.cuh", os.path.join("..", "..", "include", "spinllg.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def nvcc_path() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    cuda_lib = os.path.join(os.path.dirname(os.path.dirname(nvcc_path())), "lib64")
    cmd = [nvcc_path(), "-std=c++17", "-O3", "-lineinfo", *ARCH, "-Xcompiler", "-fPIC", "-shared",
           "-o", LIB, *[os.path.join(CSRC, f) for f in SOURCES],
           "-DSPIN_NVRTC_PATH=\"%s\"" % os.path.join(cuda_lib, "libnvrtc.so.12"), "-lcufft", "-ldl", "-Xlinker", "-rpath", "-Xlinker", cuda_lib]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
        print(" ".join(cmd))
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
