"""Builds libsable.so in-tree with nvcc for sm_100a:  python -m paper_2606_07099_b200.build [--force] [-v]"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SRC = [os.path.join(CSRC, f) for f in ("sable_capi.cu", "sable_symbolic.cpp", "sable_static.cu")]
OUT = os.path.join(HERE, "libsable.so")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "--extended-lambda",
         "-Xcompiler", "-fPIC", "-shared", "-diag-suppress", "550"]


def build(force=False, verbose=False):
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(os.path.dirname(HERE), "include", "sable.h")]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = OUT + f".{os.getpid()}.tmp"
    subprocess.check_call([nvcc] + FLAGS + os.environ.get("SABLE_NVCC_FLAGS", "").split() + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SRC)
    os.replace(tmp, OUT)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
