"""gather_probe: random 32-byte-sector gather rates of the GPU (measurement aid).

    python -m paper_1902_09396_b200.gather_probe            # prints a markdown table; needs a GPU

`build()` compiles csrc/gather_probe.cu into libhmlfc_probe.so (nvcc, sm_100a; works without a GPU).
"""
import ctypes as C
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "gather_probe.cu")
LIB = os.path.join(HERE, "libhmlfc_probe.so")
MODES = ["32-bit", "64-bit", "128-bit", "2 x 128-bit, same sector", "256-bit", "4 x 32-bit, same sector"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(SRC) > os.path.getmtime(LIB):
        subprocess.run(["/usr/local/cuda/bin/nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                        "-Xcompiler", "-fPIC", "-shared", "-cudart", "shared", "-o", LIB + ".tmp", SRC], check=True)
        os.replace(LIB + ".tmp", LIB)
    return LIB


def measure(mode: int, table_bytes: int):
    """(milliseconds, lane-gathers) of one timed launch."""
    lib = C.CDLL(build())
    lib.hmlfc_gather_probe.argtypes = [C.c_int, C.c_ulonglong, C.POINTER(C.c_float), C.POINTER(C.c_double)]
    ms, n = C.c_float(), C.c_double()
    rc = lib.hmlfc_gather_probe(mode, table_bytes, C.byref(ms), C.byref(n))
    if rc:
        raise RuntimeError(f"hmlfc_gather_probe failed with code {rc} (needs a CUDA device)")
    return ms.value, n.value


def main():
    print("| load per lane | table | ms | G sector-gathers/s | GB/s of sectors |")
    print("|---|---|---|---|---|")
    for mb in (8, 1024):
        for mode, name in enumerate(MODES):
            ms, n = measure(mode, mb << 20)
            rate = n / (ms * 1e-3) / 1e9
            print(f"| {name} | {mb} MB | {ms:.3f} | {rate:.1f} | {rate * 32:.0f} |")


if __name__ == "__main__":
    main()
