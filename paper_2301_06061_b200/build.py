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
SOURCES = ["ws_api.cu", "ws_bin.cu", "ws_grid.cu", "ws_wcorrect.cu", "ws_fft.cu", "ws_degrid.cu", "ws_probe.cu", "ws_f64.cu", "ws_static.cu"]
HEADERS = [os.path.join(CSRC, "ws_internal.h"), os.path.join(CSRC, "ws_phase.cuh"), os.path.join(CSRC, "ws_taps.cuh"), os.path.join(CSRC, "ws_place.cuh"), os.path.join(HERE, "..", "include", "wstack.h")]
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")


OBJ_DIR = os.path.join(HERE, "build")


def _newer(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """One nvcc -c per source, in parallel (objects under build/, git-ignored), then the link."""
    common = HEADERS + [os.path.abspath(__file__)]
    nvcc = os.path.join(CUDA_HOME, "bin", "nvcc")
    flags = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
             "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall"]
    if verbose:
        flags += ["-Xptxas", "-v"]
    os.makedirs(OBJ_DIR, exist_ok=True)
    jobs, objs = [], []
    for src in SOURCES:
        path, obj = os.path.join(CSRC, src), os.path.join(OBJ_DIR, src[:-3] + ".o")
        objs.append(obj)
        if force or _newer(obj, [path] + common):
            jobs.append((src, subprocess.Popen([nvcc] + flags + ["-c", path, "-o", obj])))
    for src, p in jobs:
        if p.wait() != 0:
            raise RuntimeError(f"nvcc failed on {src}")
    if force or jobs or _newer(LIB, objs):
        subprocess.run([nvcc, "-shared", "-o", LIB] + objs +
                       ["-L" + os.path.join(CUDA_HOME, "lib64"), "-lcufft", "-Xlinker",
                        "-rpath," + os.path.join(CUDA_HOME, "lib64")], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
