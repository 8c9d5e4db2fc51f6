"""Compile the CUDA library (csrc/*.cu -> libwstack.so, in-tree) for sm_100a with nvcc.

Run as `python -m paper_2301_06061_b200.build [--force]`; `build()` is also what
`__graft_entry__.build()` and the binding call.  nvcc cross-compiles without a GPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libwstack.so")
SOURCES = ["ws_api.cu", "ws_bin.cu", "ws_grid.cu", "ws_wcorrect.cu"]
HEADERS = [os.path.join(CSRC, "ws_internal.h"), os.path.join(HERE, "..", "include", "wstack.h")]
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.path.join(CUDA_HOME, "bin", "nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", "-shared", "-o", LIB]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    cmd += ["-L" + os.path.join(CUDA_HOME, "lib64"), "-lcufft", "-Xlinker", "-rpath," + os.path.join(CUDA_HOME, "lib64")]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
