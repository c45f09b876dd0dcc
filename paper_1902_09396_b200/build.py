"""Build libhmlfc_b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

Every .cu is compiled to an object under build/ (git-ignored) in parallel and only when it or a header changed; the
objects are then linked into the shared library beside this file.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
OBJ = os.path.join(HERE, "build")
SOURCES = ["hmlfc_api.cu", "hmlfc_kernels.cu", "hmlfc_decode_queue.cu", "hmlfc_search.cu", "hmlfc_hierarchy.cu", "hmlfc_encode.cu",
           "hmlfc_render_warp.cu", "hmlfc_render_cta.cu", "hmlfc_render_tiles.cu", "hmlfc_decode_rows.cu", "hmlfc_repack.cu"]
HEADERS = ["hmlfc_device.cuh", "hmlfc_kernels.cuh", "hmlfc_tables.h", "hmlfc_bise_row.cuh", "hmlfc_render_common.cuh"]
LIB = os.path.join(HERE, "libhmlfc_b200.so")

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _common_deps():
    return [os.path.join(CSRC, f) for f in HEADERS] + [os.path.join(INCLUDE, "hmlfc.h"), os.path.abspath(__file__)]


def _stale(target, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def needs_build() -> bool:
    return _stale(LIB, [os.path.join(CSRC, f) for f in SOURCES] + _common_deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    extra = os.environ.get("HMLFC_NVCC_EXTRA", "").split()   # e.g. -DHMLFC_PASS_STATS for a debugging build
    flags = NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + extra + ["-I", INCLUDE]

    def compile_one(src):
        obj = os.path.join(OBJ, src[:-3] + ".o")
        if force or extra or _stale(obj, [os.path.join(CSRC, src)] + _common_deps()):
            subprocess.run([_nvcc()] + flags + ["-c", os.path.join(CSRC, src), "-o", obj], check=True, cwd=HERE)
        return obj

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as pool:
        objs = list(pool.map(compile_one, SOURCES))
    subprocess.run([_nvcc(), "-shared", "-cudart", "shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp"] + objs, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
