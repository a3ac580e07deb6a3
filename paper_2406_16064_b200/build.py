"""Build paper_2406_16064_b200/libmm.so (sm_100a) in-tree: `python -m paper_2406_16064_b200.build`."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmm.so")
SOURCES = ["mm_lib.cu", "mm_newell_host.cpp", "mm_noalloc.cu"]
HEADERS = ["mm_fft.cuh", "mm_kernels.cuh", "mm_kernels2.cuh", "mm_passAC.cuh", "mm_passB7.cuh", "mm_passB3.cuh", "mm_passB4.cuh", "mm_llg.cuh", os.path.join("..", "..", "include", "mm.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    obj_cu = os.path.join(CSRC, "mm_lib.o")
    obj_cpp = os.path.join(CSRC, "mm_newell_host.o")
    obj_na = os.path.join(CSRC, "mm_noalloc.o")
    cmds = [
        [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "-c", os.path.join(CSRC, "mm_lib.cu"), "-o", obj_cu] + (["-Xptxas", "-v"] if verbose else []) + os.environ.get("MM_NVCC_FLAGS", "").split(),
        ["g++", "-O2", "-std=gnu++17", "-fPIC", "-c", os.path.join(CSRC, "mm_newell_host.cpp"), "-o", obj_cpp],
        [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "-c", os.path.join(CSRC, "mm_noalloc.cu"), "-o", obj_na],
        [NVCC, "-shared", "-o", LIB, obj_cu, obj_cpp, obj_na, "-lquadmath", "-lpthread"],
    ]
    for c in cmds:
        subprocess.run(c, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
