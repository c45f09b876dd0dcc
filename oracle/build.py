"""Build the HMLFC oracle (test infrastructure) into oracle/liboracle.so with gcc.

The oracle is plain C + OpenMP.  Flags that matter for parity: -ffp-contract=off (the ray
set-up must be strict IEEE fp32) and no -ffast-math.  No -march=native, so
the library built here also runs on the GPU box's host.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["colour.c", "bise.c", "encode.c", "tree.c", "stream.c", "decode.c", "render.c"]
HEADERS = ["hmlfc_oracle.h", "oracle_internal.h"]
# HMLFC_ORACLE_SANITIZE=1: the AddressSanitizer + UndefinedBehaviorSanitizer build, a second library beside
# the normal one.  A Python process that loads it needs LD_PRELOAD=$(gcc -print-file-name=libasan.so); tests/test_oracle_sanitizers.py
# re-runs the oracle pins that way in a child process.
SANITIZE = os.environ.get("HMLFC_ORACLE_SANITIZE", "") not in ("", "0")
LIB = os.path.join(HERE, "liboracle_san.so" if SANITIZE else "liboracle.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS + ["build.py"])


def build(force: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if SANITIZE else ["-O3"]
    cmd = ["gcc", "-std=c11"] + opt + ["-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB + ".tmp"] + [os.path.join(HERE, s) for s in SOURCES] + ["-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
