"""Build the host kernel emulator (tests/emu/libcales_emu.so) from the CUDA sources with nvcc, host code only."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
CSRC = os.path.join(ROOT, "paper_2411_09364_b200", "csrc")
SRC = os.path.join(HERE, "cales_emu.cu")
LIB = os.path.join(HERE, "libcales_emu.so")


def build(force=False):
    deps = [SRC, os.path.join(ROOT, "include", "cales.h")] + [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = "/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc"
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-std=c++17", "--extended-lambda", "-Xcompiler", "-fPIC",
           "-shared", "-o", LIB, SRC] + os.environ.get("CALES_NVCC_EXTRA", "").split()
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
