"""Build the CUDA product library paper_1308_1856_b200/libtdse_b200.so for sm_100a with nvcc (in-tree).

nvcc cross-compiles without a GPU.  The library links the static CUDA runtime, so loading it needs no GPU;
every compute entry point returns TDSE_ERR_CUDA when no device is present (there is no CPU fallback).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtdse_b200.so")
SOURCES = [os.path.join(CSRC, "tdse_api.cu")]
DEPS = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "tdse.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def nvcc_cmd(extra=()):
    return [NVCC, "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
            "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", *extra, "-o", LIB, *SOURCES]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = nvcc_cmd(("-Xptxas", "-v") if verbose else ())
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
