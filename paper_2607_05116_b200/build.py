"""Compile the CUDA sources under csrc/ into paper_2607_05116_b200/libcap_b200.so (sm_100a).

nvcc cross-compiles without a GPU.  -fmad=false: no implicit FMA contraction, the gate
weights and the pruning rule are defined in single IEEE fp32 operations (DESIGN.md R-S1.3).

One object per .cu file under build/ (git-ignored), compiled in parallel and rebuilt only when the
file, a header or the flags are newer; the objects are then linked into the shared library.
"""
import glob
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libcap_b200.so")
OBJ = os.path.join(HERE, "build")
SRCS = sorted(glob.glob(os.path.join(HERE, "csrc", "*.cu")))
HDRS = glob.glob(os.path.join(HERE, "csrc", "*.cuh")) + [os.path.join(ROOT, "include", "cap.h"),
                                                         os.path.abspath(__file__)]
DEPS = SRCS + HDRS

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-fmad=false", "-Xcompiler", "-fPIC", "-Xptxas", "-v",
    "-I", os.path.join(ROOT, "include"),
]


def _newer(target: str, deps) -> bool:
    return os.path.exists(target) and all(os.path.getmtime(target) >= os.path.getmtime(d) for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and _newer(LIB, DEPS):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(src: str):
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        if not force and _newer(obj, [src] + HDRS):
            return obj, None
        return obj, subprocess.run([nvcc] + NVCC_FLAGS + ["-c", "-o", obj, src], capture_output=True, text=True)

    with ThreadPoolExecutor(max_workers=min(len(SRCS), os.cpu_count() or 4)) as pool:
        done = list(pool.map(compile_one, SRCS))
    failed = False
    for obj, res in done:
        if res is not None and (verbose or res.returncode != 0):
            print(res.stdout)
            print(res.stderr)
        failed |= res is not None and res.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building libcap_b200.so")
    res = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] +
                         [o for o, _ in done], capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed linking libcap_b200.so")
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
