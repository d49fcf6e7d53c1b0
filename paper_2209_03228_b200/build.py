"""Build liblandau_b200.so in-tree with nvcc for sm_100a (no JIT cache; the .so travels with the repo snapshot)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblandau_b200.so")
SOURCES = ["landau_api.cu", "host_setup.cpp", "landau3v_api.cu", "host_setup3v.cpp", "batch_solver.cu"]
DEPS = SOURCES + ["batch_solver.hpp", "landau3v_kernels.cuh", "landau3v_dmma.cuh", "landau3v_k3.cuh", "host_setup3v.hpp", os.path.join("..", "..", "include", "landau3v.h"), "landau_kernels.cuh", "k2_gemm.cuh", "k3_ring.cuh", "k4_solve.cuh", "host_setup.hpp", "ellip_coeffs.h", os.path.join("..", "..", "include", "landau.h"),
        os.path.join("..", "..", "include", "landau_debug.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
              "-shared", "-ldl"]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force=False, verbose=False):
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + \
        [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
