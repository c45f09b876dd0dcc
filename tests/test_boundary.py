"""CPU checks of the C-ABI boundary: the library loads, exports every symbol include/hmlfc.h declares,
rejects malformed streams before touching CUDA, and refuses to compute without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def P():
    import paper_1902_09396_b200 as pkg
    from paper_1902_09396_b200 import build

    build.build()  # nvcc cross-compiles for sm_100a without a GPU
    return pkg


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "hmlfc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hmlfc_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(P):
    L = P.lib()
    declared = _declared_symbols()
    assert len(declared) >= 14
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/hmlfc.h but not exported"
    assert sorted(P.EXPORTS) == declared


def test_library_is_built_for_sm_100a(P):
    import subprocess

    out = subprocess.run(["cuobjdump", "-lelf", P.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_load_rejects_malformed_streams_with_distinct_codes(P, enc):
    cfg, lf, data, info, s = enc("cfg1_lossy")
    L = P.lib()

    def load(blob):
        buf = np.frombuffer(bytes(blob), dtype=np.uint8)
        out = C.c_void_p()
        return L.hmlfc_load(buf.ctypes.data_as(C.c_void_p), buf.size, C.byref(out)), out

    bad_magic = bytearray(data)
    bad_magic[1] ^= 0x40
    bad_version = bytearray(data)
    bad_version[4] = 9
    chroma = bytearray(data)
    chroma[49] = 2       # 0 = off, 1 = Co / Cg at half resolution (R18); anything else is not a layout this library reads
    subpel = bytearray(data)
    subpel[55] = 2       # 0 = whole-pixel motion offsets, 1 = half pixels (R28)
    subpel_flip = bytearray(data)
    subpel_flip[55] = 1  # an integer-pel stream that claims half-pel offsets: the motion strings no longer have the directory's sizes
    chroma_flip = bytearray(data)
    chroma_flip[49] = 1  # a full-resolution stream that claims subsampled chroma: its directory no longer matches its flag maps
    bad_block = bytearray(data)
    bad_block[28] = 3
    bad_dir = bytearray(data)
    off_dir = int.from_bytes(data[120:128], "little")
    bad_dir[off_dir + 8] ^= 0x01  # n_res of the first plane-channel no longer matches its flag map
    # untrusted 64-bit directory offsets near 2^64 must not wrap the bounds checks (flag map @16, payload @24, motion records @32)
    wraps = []
    for field, value in ((16, (1 << 64) - 4), (24, (1 << 64) - 32), (32, (1 << 64) - 32), (24, 1 << 63)):
        w = bytearray(data)
        w[off_dir + 48 + field:off_dir + 48 + field + 8] = value.to_bytes(8, "little")   # second entry: a plane-channel with blocks
        wraps.append((w, -6))
    cases = [(bad_magic, -1), (data[:6], -2), (data[:100], -2), (data[:len(data) // 2], -2), (bad_version, -3),
             (chroma, -5), (chroma_flip, -6), (subpel, -5), (subpel_flip, -6), (bad_block, -5), (bad_dir, -6)] + wraps
    for blob, code in cases:
        rc, out = load(blob)
        assert rc == code and not out.value, (rc, code)
    assert L.hmlfc_load(None, 0, None) == -4
    assert b"magic" in L.hmlfc_strerror(-1) and b"truncated" in L.hmlfc_strerror(-2)


def test_entry_points_validate_arguments(P):
    L = P.lib()
    assert L.hmlfc_decode(None, None, 0, None, None) == -4
    assert L.hmlfc_render(None, None, 0, 1, 1, None, None) == -4
    assert L.hmlfc_info(None, None) == -4
    L.hmlfc_free(None)  # no-op
    assert L.hmlfc_search(None, None, 1, 8, 8, 4, 1, None, None) == -4      # null pointers
    assert L.hmlfc_search(None, None, 0, 8, 8, 3, 1, None, None) == -5      # block does not divide the image
    assert L.hmlfc_search(None, None, 0, 8, 8, 4, 65, None, None) == -5     # window > 64
    assert L.hmlfc_search(None, None, 0, 8, 8, 4, 16, None, None) == 0      # nothing to do
    assert L.hmlfc_hierarchy(None, 2, 2, 8, 8, 1, None, None, None) == -4
    assert P.hmlfc_hierarchy_sizes(17, 17, 3) == (17 * 17 + 9 * 9 + 5 * 5, 9 * 9 + 5 * 5 + 3 * 3)   # 17 -> 9 -> 5 -> 3 (R3)
    assert P.hmlfc_hierarchy_sizes(16, 16, 3) == (256 + 64 + 16, 64 + 16 + 4)
    # hmlfc_encode checks its arguments before any CUDA call
    out, n = C.c_void_p(), C.c_size_t()
    p = P.EncodeParams()
    p.U, p.V, p.Ws, p.Ht, p.height, p.block, p.window = 2, 2, 16, 16, 1, 4, 4
    dummy = C.c_void_p(16)
    assert L.hmlfc_encode(None, C.byref(p), C.byref(out), C.byref(n), None, None) == -4     # null light field
    p.block = 3
    assert L.hmlfc_encode(dummy, C.byref(p), C.byref(out), C.byref(n), None, None) == -5    # B not in {2, 4, 8}
    p.block, p.Ws = 4, 18
    assert L.hmlfc_encode(dummy, C.byref(p), C.byref(out), C.byref(n), None, None) == -5    # B does not divide Ws
    p.Ws, p.policy = 16, 4
    assert L.hmlfc_encode(dummy, C.byref(p), C.byref(out), C.byref(n), None, None) == -4    # unknown policy
    L.hmlfc_stream_free(None)  # no-op


def test_no_cpu_fallback(P, enc):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    cfg, lf, data, info, s = enc("cfg1_lossy")
    with pytest.raises(P.HmlfcError):
        P.hmlfc_load(data)
