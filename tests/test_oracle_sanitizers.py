"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (ASan/UBSan build of the CPU code).

oracle/build.py builds a second library (liboracle_san.so, -fsanitize=address,undefined, UBSan not recovering) when
HMLFC_ORACLE_SANITIZE=1; a child Python process with libasan preloaded re-runs the oracle's pins against it.  Any
out-of-bounds access, use after free, signed overflow or misaligned access in the encoder, the stream writer / parser,
the three decoders, the renderer or the byte counter aborts the child."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SUITE = ["tests/test_oracle_colour_bise.py", "tests/test_oracle_tree.py", "tests/test_oracle_codec.py", "tests/test_oracle_render.py",
         "tests/test_golden.py"]


def test_oracle_pins_pass_under_asan_and_ubsan():
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan is not installed with this gcc")
    env = dict(os.environ, HMLFC_ORACLE_SANITIZE="1", LD_PRELOAD=asan, OMP_NUM_THREADS="4",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    # the exhaustive 2^24 colour round trip and the full-size cfg1 encodes are covered by the normal build; the sanitizer build (~10x
    # slower) runs everything else
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "-k",
                        "not exhaustive and not cfg1 and not sanitizers"] + SUITE, cwd=ROOT, env=env, capture_output=True, text=True)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "passed" in r.stdout
