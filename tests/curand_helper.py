"""Builds the cuRAND cross-check helper of tests/test_gpu_curand.py (curand_philox_check.cu -> a small shared library).

A plain module on purpose: no pytest, no oracle, no product imports, so that __graft_entry__.build() can compile the helper
(one more .cu for sm_100a) on a machine that has neither pytest nor a GPU.  Test infrastructure only.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "curand_philox_check.cu")
LIB = os.path.join(HERE, "build", "libcurand_philox_check.so")


def build_helper(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        os.makedirs(os.path.dirname(LIB), exist_ok=True)
        nvcc = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
        subprocess.run([nvcc, "-O2", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC",
                        "-shared", "-cudart", "static", "-o", LIB, SRC], check=True)
    return LIB
