"""Builds the test-only CUDA helpers (in-tree, so the .so travels to the GPU box)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libphilox_curand.so")


def build(force=False):
    src = os.path.join(HERE, "philox_curand.cu")
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(src):
        return LIB
    subprocess.run([os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"), "-O2", "-gencode", "arch=compute_100a,code=sm_100a",
                    "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "-o", LIB, src], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
