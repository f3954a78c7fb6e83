"""Build libspshell.so in-tree: nvcc (sm_100a) for the CUDA translation unit, g++ for the host
matrix construction (binary128 via libquadmath)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libspshell.so")
SOURCES = ["spshell.cu", "host_build.cpp", "sp_device.cuh", "sp_internal.h", "kernels_gemm.cuh", "kernels_gemm2.cuh", "kernels_gradphi.cuh", "kernels_theta2.cuh", "kernels_grad.cuh",
           "kernels_filter.cuh", "kernels_fused.cuh", "kernels_wave.cuh", "kernels_ghg.cuh"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES] + [os.path.join(HERE, "..", "include", "spshell.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    obj_host = os.path.join(CSRC, "host_build.o")
    obj_cu = os.path.join(CSRC, "spshell.o")
    subprocess.run(["g++", "-O2", "-std=gnu++17", "-fPIC", "-c", os.path.join(CSRC, "host_build.cpp"), "-o", obj_host], check=True)
    cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
           "-c", os.path.join(CSRC, "spshell.cu"), "-o", obj_cu]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.run(cmd, check=True)
    subprocess.run([NVCC, "-shared", "-o", LIB, obj_cu, obj_host, "-lquadmath", "-lpthread", "-lcudart"], check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
