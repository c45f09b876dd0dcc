"""Thin Python binding of libhmlfc_b200.so (include/hmlfc.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing, or a call needs
a GPU and none is present, the call raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhmlfc_b200.so")

# every symbol include/hmlfc.h declares
EXPORTS = (
    "hmlfc_load", "hmlfc_info", "hmlfc_decode", "hmlfc_decode_views", "hmlfc_decode_blocks", "hmlfc_render", "hmlfc_render_noalloc", "hmlfc_render_lod", "hmlfc_lod_levels", "hmlfc_decode_host", "hmlfc_decode_views_host", "hmlfc_render_host",
    "hmlfc_last_oob_count", "hmlfc_footprint_render", "hmlfc_footprint_decode", "hmlfc_set_render_variant", "hmlfc_set_decode_variant", "hmlfc_search", "hmlfc_hierarchy", "hmlfc_hierarchy_sizes", "hmlfc_set_min_level", "hmlfc_encode", "hmlfc_encode_psnr", "hmlfc_stream_free", "hmlfc_encode_release_scratch",
    "hmlfc_launch_count", "hmlfc_free", "hmlfc_strerror", "hmlfc_last_cuda_error",
)

RENDER_AUTO, RENDER_PIXEL, RENDER_WARP, RENDER_WARP8, RENDER_CTA, RENDER_CTA_BIG, RENDER_CTA_SMALL = 0, 1, 4, 5, 6, 7, 8
RENDER_CTA_1024, RENDER_CTA_512, RENDER_TILES, RENDER_TILES4, RENDER_TILES_W512, RENDER_TILES_W256, RENDER_TILES_W256X3 = 9, 10, 11, 12, 13, 14, 15
# every configuration of the two fused kernels for 4 x 4 blocks (all give the same bytes; hmlfc_set_render_variant forces one)
RENDER_FUSED = (RENDER_CTA, RENDER_CTA_BIG, RENDER_CTA_SMALL, RENDER_CTA_1024, RENDER_CTA_512, RENDER_TILES, RENDER_TILES4,
                RENDER_TILES_W512, RENDER_TILES_W256, RENDER_TILES_W256X3)
DECODE_AUTO, DECODE_THREAD, DECODE_QUEUE, DECODE_QUEUE_LAZY, DECODE_QUEUE_BLOCKREC = 0, 1, 2, 3, 4


class HmlfcError(RuntimeError):
    def __init__(self, code, what, detail=""):
        super().__init__(f"{what}: {detail or code} (code {code})")
        self.code = code


class Info(C.Structure):
    _fields_ = [
        ("U", C.c_int32), ("V", C.c_int32), ("Ws", C.c_int32), ("Ht", C.c_int32),
        ("height", C.c_int32), ("block", C.c_int32), ("window", C.c_int32),
        ("tau_ref", C.c_int32), ("tau_res", C.c_int32),
        ("uv_origin", C.c_float * 2), ("uv_step", C.c_float * 2), ("st_origin", C.c_float * 2),
        ("st_step", C.c_float * 2), ("z_st", C.c_float),
        ("background", C.c_uint8 * 3), ("_pad", C.c_uint8),
        ("stream_bytes", C.c_uint64), ("device_bytes", C.c_uint64), ("n_plane_channels", C.c_uint64),
    ]


class Footprint(C.Structure):
    _fields_ = [
        ("blocks_touched", C.c_int64), ("flag_bits", C.c_int64), ("payload_bits15", C.c_int64),
        ("mv_bits15", C.c_int64), ("rkv_bytes", C.c_int64), ("out_bytes", C.c_int64), ("in_bytes", C.c_int64),
        ("bytes_alg", C.c_double),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib():
    """Load the CUDA library; fail loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise HmlfcError(-1, "libhmlfc_b200.so not built",
                         f"{LIB_PATH} is missing; run `python -m paper_1902_09396_b200.build` (there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64 = C.c_void_p, C.c_int64
    L.hmlfc_load.argtypes, L.hmlfc_load.restype = [vp, C.c_size_t, C.POINTER(vp)], C.c_int
    L.hmlfc_info.argtypes, L.hmlfc_info.restype = [vp, C.POINTER(Info)], C.c_int
    L.hmlfc_decode.argtypes, L.hmlfc_decode.restype = [vp, vp, i64, vp, vp], C.c_int
    L.hmlfc_decode_views.argtypes, L.hmlfc_decode_views.restype = [vp, vp, i64, vp, vp], C.c_int
    L.hmlfc_decode_blocks.argtypes, L.hmlfc_decode_blocks.restype = [vp, vp, i64, vp, vp], C.c_int
    L.hmlfc_render.argtypes, L.hmlfc_render.restype = [vp, vp, C.c_int, C.c_int, C.c_int, vp, vp], C.c_int
    L.hmlfc_render_noalloc.argtypes, L.hmlfc_render_noalloc.restype = [vp, vp, C.c_int, C.c_int, C.c_int, vp, vp], C.c_int
    L.hmlfc_render_lod.argtypes, L.hmlfc_render_lod.restype = [vp, vp, vp, C.c_int, C.c_int, C.c_int, vp, vp], C.c_int
    L.hmlfc_lod_levels.argtypes, L.hmlfc_lod_levels.restype = [vp, vp, C.c_int, C.c_float, vp], C.c_int
    L.hmlfc_decode_host.argtypes, L.hmlfc_decode_host.restype = [vp, vp, i64, vp], C.c_int
    L.hmlfc_decode_views_host.argtypes, L.hmlfc_decode_views_host.restype = [vp, vp, i64, vp], C.c_int
    L.hmlfc_render_host.argtypes, L.hmlfc_render_host.restype = [vp, vp, C.c_int, C.c_int, C.c_int, vp], C.c_int
    L.hmlfc_last_oob_count.argtypes, L.hmlfc_last_oob_count.restype = [vp, C.POINTER(i64)], C.c_int
    L.hmlfc_footprint_render.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, C.POINTER(Footprint)]
    L.hmlfc_footprint_render.restype = C.c_int
    L.hmlfc_footprint_decode.argtypes, L.hmlfc_footprint_decode.restype = [vp, vp, i64, C.POINTER(Footprint)], C.c_int
    L.hmlfc_set_render_variant.argtypes, L.hmlfc_set_render_variant.restype = [vp, C.c_int], C.c_int
    L.hmlfc_set_decode_variant.argtypes, L.hmlfc_set_decode_variant.restype = [vp, C.c_int], C.c_int
    L.hmlfc_set_min_level.argtypes, L.hmlfc_set_min_level.restype = [vp, C.c_int], C.c_int
    L.hmlfc_search.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp, vp]
    L.hmlfc_search.restype = C.c_int
    L.hmlfc_hierarchy_sizes.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(i64), C.POINTER(i64)]
    L.hmlfc_hierarchy_sizes.restype = C.c_int
    L.hmlfc_hierarchy.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp, vp, vp]
    L.hmlfc_hierarchy.restype = C.c_int
    L.hmlfc_launch_count.argtypes, L.hmlfc_launch_count.restype = [vp, C.POINTER(i64)], C.c_int
    L.hmlfc_encode.argtypes = [vp, vp, C.POINTER(vp), C.POINTER(C.c_size_t), vp, vp]
    L.hmlfc_encode.restype = C.c_int
    L.hmlfc_stream_free.argtypes, L.hmlfc_stream_free.restype = [vp], None
    L.hmlfc_encode_psnr.argtypes = [vp, vp, C.c_double, C.c_double, C.c_int, C.POINTER(vp), C.POINTER(C.c_size_t), vp, vp]
    L.hmlfc_encode_psnr.restype = C.c_int
    L.hmlfc_encode_release_scratch.argtypes, L.hmlfc_encode_release_scratch.restype = [], C.c_int
    L.hmlfc_free.argtypes, L.hmlfc_free.restype = [vp], None
    L.hmlfc_strerror.argtypes, L.hmlfc_strerror.restype = [C.c_int], C.c_char_p
    L.hmlfc_last_cuda_error.argtypes, L.hmlfc_last_cuda_error.restype = [vp], C.c_int
    _lib = L
    return L


def _check(rc, what, handle=None):
    if rc != 0:
        detail = lib().hmlfc_strerror(rc).decode()
        if handle is not None and rc == -8:
            detail += f" (cudaError {lib().hmlfc_last_cuda_error(handle)})"
        raise HmlfcError(rc, what, detail)


def _require_cuda():
    import torch

    if not torch.cuda.is_available():
        raise HmlfcError(-8, "no CUDA device", "the HMLFC hot path runs only on the GPU (there is no CPU fallback)")
    return torch


def _stream_ptr(stream):
    torch = _require_cuda()
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


class Handle:
    """Owns one loaded stream on the current CUDA device."""

    def __init__(self, ptr):
        self._h = ptr
        self.info = Info()
        _check(lib().hmlfc_info(self._h, C.byref(self.info)), "hmlfc_info")

    def free(self):
        if self._h:
            lib().hmlfc_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def hmlfc_load(stream_bytes: bytes) -> Handle:
    """Upload a serialized HMLFC stream to the current CUDA device (include/hmlfc.h: hmlfc_load)."""
    _require_cuda().cuda.current_device()  # make sure a context exists on the current device
    buf = np.frombuffer(stream_bytes, dtype=np.uint8)
    out = C.c_void_p()
    _check(lib().hmlfc_load(buf.ctypes.data_as(C.c_void_p), buf.size, C.byref(out)), "hmlfc_load")
    return Handle(out)


def hmlfc_decode(h: Handle, coords, out=None, stream=None):
    """coords: CUDA int32 tensor [n][4] = (u,v,s,t); returns CUDA uint8 tensor [n][3]."""
    torch = _require_cuda()
    assert coords.is_cuda and coords.dtype == torch.int32 and coords.is_contiguous() and coords.shape[-1] == 4
    n = coords.numel() // 4
    if out is None:
        out = torch.empty((n, 3), dtype=torch.uint8, device=coords.device)
    assert out.is_cuda and out.dtype == torch.uint8 and out.is_contiguous() and out.numel() == 3 * n
    _check(lib().hmlfc_decode(h._h, C.c_void_p(coords.data_ptr()), n, C.c_void_p(out.data_ptr()), _stream_ptr(stream)),
           "hmlfc_decode", h._h)
    return out


def hmlfc_decode_views(h: Handle, views, out=None, stream=None):
    """views: CUDA int32 tensor [n][2] = (u,v); returns CUDA uint8 tensor [n][Ht][Ws][3] (every pixel of every listed view)."""
    torch = _require_cuda()
    assert views.is_cuda and views.dtype == torch.int32 and views.is_contiguous() and views.shape[-1] == 2
    n = views.numel() // 2
    Ht, Ws = h.info.Ht, h.info.Ws
    if out is None:
        out = torch.empty((n, Ht, Ws, 3), dtype=torch.uint8, device=views.device)
    assert out.is_cuda and out.dtype == torch.uint8 and out.is_contiguous() and out.numel() == n * Ht * Ws * 3
    _check(lib().hmlfc_decode_views(h._h, C.c_void_p(views.data_ptr()), n, C.c_void_p(out.data_ptr()), _stream_ptr(stream)),
           "hmlfc_decode_views", h._h)
    return out


def hmlfc_decode_blocks(h: Handle, blocks, out=None, stream=None):
    """blocks: CUDA int32 tensor [n][4] = (u,v,bx,by); returns CUDA uint8 tensor [n][B][B][3]."""
    torch = _require_cuda()
    assert blocks.is_cuda and blocks.dtype == torch.int32 and blocks.is_contiguous() and blocks.shape[-1] == 4
    n, B = blocks.numel() // 4, h.info.block
    if out is None:
        out = torch.empty((n, B, B, 3), dtype=torch.uint8, device=blocks.device)
    assert out.is_cuda and out.dtype == torch.uint8 and out.is_contiguous() and out.numel() == n * B * B * 3
    _check(lib().hmlfc_decode_blocks(h._h, C.c_void_p(blocks.data_ptr()), n, C.c_void_p(out.data_ptr()), _stream_ptr(stream)),
           "hmlfc_decode_blocks", h._h)
    return out


def hmlfc_render(h: Handle, cameras, W: int, H: int, out=None, stream=None):
    """cameras: CUDA float32 tensor [n_views][16]; returns CUDA uint8 tensor [n_views][H][W][3]."""
    torch = _require_cuda()
    assert cameras.is_cuda and cameras.dtype == torch.float32 and cameras.is_contiguous() and cameras.shape[-1] == 16
    n = cameras.numel() // 16
    if out is None:
        out = torch.empty((n, H, W, 3), dtype=torch.uint8, device=cameras.device)
    assert out.is_cuda and out.dtype == torch.uint8 and out.is_contiguous() and out.numel() == n * H * W * 3
    _check(lib().hmlfc_render(h._h, C.c_void_p(cameras.data_ptr()), n, W, H, C.c_void_p(out.data_ptr()), _stream_ptr(stream)),
           "hmlfc_render", h._h)
    return out


NOALLOC_MAX_TILES = 4096   # include/hmlfc.h: HMLFC_NOALLOC_MAX_TILES


def hmlfc_render_noalloc(h: Handle, cameras, W: int, H: int, out, stream=None):
    """hmlfc_render with the tile tables in the library's static device buffer: the call allocates nothing (the caller passes `out`).
    At most NOALLOC_MAX_TILES tiles per call (HmlfcError -9 beyond); calls that overlap on the GPU race on the buffer."""
    torch = _require_cuda()
    assert cameras.is_cuda and cameras.dtype == torch.float32 and cameras.is_contiguous() and cameras.shape[-1] == 16
    n = cameras.numel() // 16
    assert out.is_cuda and out.dtype == torch.uint8 and out.is_contiguous() and out.numel() == n * H * W * 3
    _check(lib().hmlfc_render_noalloc(h._h, C.c_void_p(cameras.data_ptr()), n, W, H, C.c_void_p(out.data_ptr()), _stream_ptr(stream)),
           "hmlfc_render_noalloc", h._h)
    return out


def hmlfc_render_lod(h: Handle, cameras, levels: np.ndarray, W: int, H: int, out=None, stream=None):
    """Per-view level of detail: cameras as for hmlfc_render, levels = HOST int32 [n_views] (numpy)."""
    torch = _require_cuda()
    assert cameras.is_cuda and cameras.dtype == torch.float32 and cameras.is_contiguous() and cameras.shape[-1] == 16
    n = cameras.numel() // 16
    levels = np.ascontiguousarray(levels, dtype=np.int32)
    assert levels.shape == (n,)
    if out is None:
        out = torch.empty((n, H, W, 3), dtype=torch.uint8, device=cameras.device)
    assert out.is_cuda and out.dtype == torch.uint8 and out.is_contiguous() and out.numel() == n * H * W * 3
    _check(lib().hmlfc_render_lod(h._h, C.c_void_p(cameras.data_ptr()), levels.ctypes.data_as(C.c_void_p), n, W, H,
                                  C.c_void_p(out.data_ptr()), _stream_ptr(stream)), "hmlfc_render_lod", h._h)
    return out


def hmlfc_lod_levels(h: Handle, cameras: np.ndarray, d0: float) -> np.ndarray:
    """The distance rule: HOST float32 [n_views][16] -> int32 [n_views] = floor(log2(|z_st - eye.z| / d0)) in [0, height]."""
    cameras = np.ascontiguousarray(cameras, dtype=np.float32).reshape(-1, 16)
    out = np.empty(cameras.shape[0], dtype=np.int32)
    _check(lib().hmlfc_lod_levels(h._h, cameras.ctypes.data_as(C.c_void_p), cameras.shape[0], C.c_float(d0), out.ctypes.data_as(C.c_void_p)),
           "hmlfc_lod_levels", h._h)
    return out


def hmlfc_decode_host(h: Handle, coords: np.ndarray, out: np.ndarray = None) -> np.ndarray:
    """End-to-end decode with HOST buffers (numpy, ideally backed by pinned memory)."""
    _require_cuda()
    assert coords.dtype == np.int32 and coords.flags.c_contiguous and coords.shape[-1] == 4
    n = coords.size // 4
    if out is None:
        out = np.empty((n, 3), dtype=np.uint8)
    assert out.dtype == np.uint8 and out.flags.c_contiguous and out.size == 3 * n
    _check(lib().hmlfc_decode_host(h._h, coords.ctypes.data_as(C.c_void_p), n, out.ctypes.data_as(C.c_void_p)),
           "hmlfc_decode_host", h._h)
    return out


def hmlfc_decode_views_host(h: Handle, views: np.ndarray, out: np.ndarray = None) -> np.ndarray:
    """End-to-end dense decode with HOST buffers: views int32 [n][2] = (u,v) -> uint8 [n][Ht][Ws][3]."""
    _require_cuda()
    assert views.dtype == np.int32 and views.flags.c_contiguous and views.shape[-1] == 2
    n = views.size // 2
    Ht, Ws = h.info.Ht, h.info.Ws
    if out is None:
        out = np.empty((n, Ht, Ws, 3), dtype=np.uint8)
    assert out.dtype == np.uint8 and out.flags.c_contiguous and out.size == n * Ht * Ws * 3
    _check(lib().hmlfc_decode_views_host(h._h, views.ctypes.data_as(C.c_void_p), n, out.ctypes.data_as(C.c_void_p)),
           "hmlfc_decode_views_host", h._h)
    return out


def hmlfc_render_host(h: Handle, cameras: np.ndarray, W: int, H: int, out: np.ndarray = None) -> np.ndarray:
    """End-to-end render with HOST buffers (numpy, ideally backed by pinned memory)."""
    _require_cuda()
    assert cameras.dtype == np.float32 and cameras.flags.c_contiguous and cameras.shape[-1] == 16
    n = cameras.size // 16
    if out is None:
        out = np.empty((n, H, W, 3), dtype=np.uint8)
    assert out.dtype == np.uint8 and out.flags.c_contiguous and out.size == n * H * W * 3
    _check(lib().hmlfc_render_host(h._h, cameras.ctypes.data_as(C.c_void_p), n, W, H, out.ctypes.data_as(C.c_void_p)),
           "hmlfc_render_host", h._h)
    return out


def hmlfc_last_oob_count(h: Handle) -> int:
    v = C.c_int64()
    _check(lib().hmlfc_last_oob_count(h._h, C.byref(v)), "hmlfc_last_oob_count", h._h)
    return v.value


def hmlfc_footprint_render(h: Handle, cameras, W: int, H: int) -> dict:
    torch = _require_cuda()
    assert cameras.is_cuda and cameras.dtype == torch.float32 and cameras.is_contiguous()
    fp = Footprint()
    torch.cuda.synchronize()
    _check(lib().hmlfc_footprint_render(h._h, C.c_void_p(cameras.data_ptr()), cameras.numel() // 16, W, H, C.byref(fp)),
           "hmlfc_footprint_render", h._h)
    return fp.as_dict()


def hmlfc_footprint_decode(h: Handle, coords) -> dict:
    torch = _require_cuda()
    assert coords.is_cuda and coords.dtype == torch.int32 and coords.is_contiguous()
    fp = Footprint()
    torch.cuda.synchronize()
    _check(lib().hmlfc_footprint_decode(h._h, C.c_void_p(coords.data_ptr()), coords.numel() // 4, C.byref(fp)),
           "hmlfc_footprint_decode", h._h)
    return fp.as_dict()


def hmlfc_set_render_variant(h: Handle, variant: int):
    _check(lib().hmlfc_set_render_variant(h._h, variant), "hmlfc_set_render_variant")


def hmlfc_set_min_level(h: Handle, min_level: int):
    _check(lib().hmlfc_set_min_level(h._h, min_level), "hmlfc_set_min_level")


def hmlfc_set_decode_variant(h: Handle, variant: int):
    _check(lib().hmlfc_set_decode_variant(h._h, variant), "hmlfc_set_decode_variant")


def hmlfc_search(planes, pairs, block: int, window: int, out=None, stream=None):
    """planes: cuda int16 [n_planes][Ht][Ws]; pairs: cuda int32 [n_pairs][2]; returns cuda int32 [n_pairs][Ht/B][Ws/B][4]."""
    torch = _require_cuda()
    assert planes.is_cuda and planes.dtype == torch.int16 and planes.is_contiguous() and planes.dim() == 3
    assert pairs.is_cuda and pairs.dtype == torch.int32 and pairs.is_contiguous() and pairs.dim() == 2 and pairs.shape[1] == 2
    n_pairs, Ht, Ws = int(pairs.shape[0]), int(planes.shape[1]), int(planes.shape[2])
    if out is None:
        out = torch.empty((n_pairs, Ht // max(block, 1), Ws // max(block, 1), 4), dtype=torch.int32, device=planes.device)
    assert out.is_cuda and out.dtype == torch.int32 and out.is_contiguous()
    st = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().hmlfc_search(C.c_void_p(planes.data_ptr()), C.c_void_p(pairs.data_ptr()), n_pairs, Ws, Ht, block, window,
                              C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream)), "hmlfc_search")
    return out


def hmlfc_hierarchy_sizes(U: int, V: int, height: int):
    """(n_srv_planes, n_x_planes) per channel."""
    a, b = C.c_int64(), C.c_int64()
    _check(lib().hmlfc_hierarchy_sizes(U, V, height, C.byref(a), C.byref(b)), "hmlfc_hierarchy_sizes")
    return a.value, b.value


def hmlfc_hierarchy(lf, height: int, srv=None, x=None, stream=None):
    """lf: cuda uint8 [V][U][Ht][Ws][3]; returns (srv int16 [3][n_srv][Ht][Ws], x int16 [3][n_x][Ht][Ws]) on the device."""
    torch = _require_cuda()
    assert lf.is_cuda and lf.dtype == torch.uint8 and lf.is_contiguous() and lf.dim() == 5 and lf.shape[4] == 3
    V, U, Ht, Ws = (int(v) for v in lf.shape[:4])
    ns, nx = hmlfc_hierarchy_sizes(U, V, height)
    if srv is None:
        srv = torch.empty((3, ns, Ht, Ws), dtype=torch.int16, device=lf.device)
    if x is None:
        x = torch.empty((3, nx, Ht, Ws), dtype=torch.int16, device=lf.device)
    assert srv.is_cuda and srv.dtype == torch.int16 and srv.is_contiguous() and tuple(srv.shape) == (3, ns, Ht, Ws)
    assert x.is_cuda and x.dtype == torch.int16 and x.is_contiguous() and tuple(x.shape) == (3, nx, Ht, Ws)
    st = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().hmlfc_hierarchy(C.c_void_p(lf.data_ptr()), U, V, Ws, Ht, height, C.c_void_p(srv.data_ptr()),
                                 C.c_void_p(x.data_ptr()), C.c_void_p(st.cuda_stream)), "hmlfc_hierarchy")
    return srv, x


class EncodeParams(C.Structure):
    _fields_ = [("U", C.c_int32), ("V", C.c_int32), ("Ws", C.c_int32), ("Ht", C.c_int32), ("height", C.c_int32),
                ("block", C.c_int32), ("window", C.c_int32), ("tau_ref", C.c_int32), ("tau_res", C.c_int32), ("policy", C.c_int32),
                ("uv_origin", C.c_float * 2), ("uv_step", C.c_float * 2), ("st_origin", C.c_float * 2), ("st_step", C.c_float * 2),
                ("z_st", C.c_float), ("background", C.c_ubyte * 3), ("_pad", C.c_ubyte), ("seed", C.c_uint64)]


class EncodeStats(C.Structure):
    _fields_ = [("ms_hierarchy", C.c_float), ("ms_search", C.c_float), ("ms_classify", C.c_float), ("ms_pack", C.c_float),
                ("ms_wall", C.c_float), ("ms_assemble", C.c_float),
                ("n_plane_channels", C.c_int64), ("n_res_blocks", C.c_int64), ("n_pred_blocks", C.c_int64),
                ("n_search_blocks", C.c_int64), ("kernel_launches", C.c_int32), ("cuda_error", C.c_int32),
                ("sse", C.c_int64), ("psnr", C.c_double), ("tau_ref", C.c_int32), ("tau_res", C.c_int32),
                ("bisection_steps", C.c_int32), ("_pad", C.c_int32)]


def hmlfc_encode(lf, height: int, block: int = 4, window: int = 16, tau_ref: int = 0, tau_res: int = 0, policy: int = 0,
                 geometry: dict = None, background=(0, 0, 0), seed: int = 0, stream=None, target_psnr: float = None,
                 tol: float = 0.25, max_iter: int = 12):
    """lf: cuda uint8 [V][U][Ht][Ws][3].  Returns (stream bytes, stats dict): the whole encoder runs in CUDA kernels, the host
    only lays out the sections.  geometry: dict(uv_origin, uv_step, st_origin, st_step, z_st) or None for the unit slab.
    target_psnr: let hmlfc_encode_psnr choose the thresholds by bisection (tau_ref / tau_res are then ignored)."""
    torch = _require_cuda()
    assert lf.is_cuda and lf.dtype == torch.uint8 and lf.is_contiguous() and lf.dim() == 5 and lf.shape[4] == 3
    p = EncodeParams()
    p.V, p.U, p.Ht, p.Ws = (int(v) for v in lf.shape[:4])
    p.height, p.block, p.window, p.tau_ref, p.tau_res, p.policy = height, block, window, tau_ref, tau_res, policy
    g = geometry or dict(uv_origin=(0.0, 0.0), uv_step=(1.0, 1.0), st_origin=(0.0, 0.0), st_step=(1.0, 1.0), z_st=1.0)
    for k in ("uv_origin", "uv_step", "st_origin", "st_step"):
        getattr(p, k)[0], getattr(p, k)[1] = float(g[k][0]), float(g[k][1])
    p.z_st = float(g["z_st"])
    for i in range(3):
        p.background[i] = background[i]
    p.seed = seed
    out, n, stats = C.c_void_p(), C.c_size_t(), EncodeStats()
    st = stream if stream is not None else torch.cuda.current_stream()
    if target_psnr is None:
        rc = lib().hmlfc_encode(C.c_void_p(lf.data_ptr()), C.byref(p), C.byref(out), C.byref(n), C.byref(stats), C.c_void_p(st.cuda_stream))
    else:
        rc = lib().hmlfc_encode_psnr(C.c_void_p(lf.data_ptr()), C.byref(p), float(target_psnr), float(tol), int(max_iter), C.byref(out),
                                     C.byref(n), C.byref(stats), C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise HmlfcError(rc, "hmlfc_encode", f"{lib().hmlfc_strerror(rc).decode()} (cuda error {stats.cuda_error})")
    try:
        data = C.string_at(out, n.value)
    finally:
        lib().hmlfc_stream_free(out)
    return data, {k: getattr(stats, k) for k, _ in EncodeStats._fields_ if k != "_pad"}


def hmlfc_encode_release_scratch():
    _check(lib().hmlfc_encode_release_scratch(), "hmlfc_encode_release_scratch")


def hmlfc_launch_count(h: Handle) -> int:
    v = C.c_int64()
    _check(lib().hmlfc_launch_count(h._h, C.byref(v)), "hmlfc_launch_count")
    return v.value


def hmlfc_free(h: Handle):
    h.free()
