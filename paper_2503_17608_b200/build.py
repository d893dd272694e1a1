"""Build libcelstep.so (the C-ABI CUDA library, include/cel.h) in-tree for sm_100a with nvcc."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcelstep.so")
SOURCES = ["cel_api.cu", "cel_noalloc.cu"]
DEPS = ["cel_api.cu", "cel_noalloc.cu", "cel_kernels.cuh", "cel_physics.cuh", "cel_tail.cuh", "cel_device.cuh", os.path.join("..", "..", "include", "cel.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-fmad=false", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(os.path.join(CSRC, d)) <= t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = ["-DCEL_NVTX"] if os.environ.get("CEL_NVTX") == "1" else []   # NVTX ranges per phase (compile-time switch)
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
