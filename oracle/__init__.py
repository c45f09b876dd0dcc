"""ctypes binding to the HMLFC oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  The CUDA path (paper_1902_09396_b200) never does.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

POLICY_ADAPTIVE, POLICY_ALL, POLICY_LITERAL, POLICY_NOMOTION = 0, 1, 2, 3
BISE_PLAIN, BISE_TRIT, BISE_QUINT = 0, 1, 2
E_MAGIC, E_TRUNCATED, E_VERSION, E_PARAM, E_NOMEM, E_CORRUPT = -1, -2, -3, -4, -5, -6


class Params(C.Structure):
    _fields_ = [
        ("U", C.c_int32), ("V", C.c_int32), ("Ws", C.c_int32), ("Ht", C.c_int32),
        ("height", C.c_int32), ("block", C.c_int32), ("window", C.c_int32),
        ("tau_ref", C.c_int32), ("tau_res", C.c_int32), ("policy", C.c_int32), ("nthreads", C.c_int32),
        ("uv_origin", C.c_float * 2), ("uv_step", C.c_float * 2),
        ("st_origin", C.c_float * 2), ("st_step", C.c_float * 2), ("z_st", C.c_float),
        ("background", C.c_uint8 * 3), ("chroma", C.c_uint8), ("subpel", C.c_uint8), ("seed", C.c_uint64),
    ]


class Stats(C.Structure):
    _fields_ = [
        ("taps", C.c_int64), ("blocks_touched", C.c_int64), ("flag_bits", C.c_int64),
        ("payload_bits15", C.c_int64), ("mv_bits15", C.c_int64), ("rkv_bytes", C.c_int64),
        ("out_bytes", C.c_int64), ("in_bytes", C.c_int64), ("bytes_alg", C.c_double),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp, i32, i64, u32, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64
    pi32 = C.POINTER(C.c_int32)
    sig = {
        "orc_rgb_to_ycocg": (None, [C.c_int] * 3 + [C.POINTER(C.c_int)] * 3),
        "orc_ycocg_to_rgb": (None, [C.c_int] * 3 + [C.POINTER(C.c_int)] * 3),
        "orc_colour_roundtrip_failures": (i64, []),
        "orc_bise_choose": (None, [u32, pi32, pi32]),
        "orc_bise_nbits": (u64, [u32, u64]),
        "orc_bise_encode": (C.c_int, [vp, u64, u32, vp]),
        "orc_bise_decode_at": (u32, [vp, u32, u64]),
        "orc_bise_decode_seq": (None, [vp, u32, u64, vp]),
        "orc_encode_begin": (vp, [vp, C.POINTER(Params), C.POINTER(C.c_int)]),
        "orc_tree_threshold": (C.c_int, [vp, C.c_int, C.c_int, C.c_int]),
        "orc_tree_serialize": (i64, [vp, C.POINTER(vp)]),
        "orc_tree_reconstruct": (C.c_int, [vp, vp]),
        "orc_tree_free": (None, [vp]),
        "orc_free": (None, [vp]),
        "orc_tree_level_dims": (C.c_int, [vp, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]),
        "orc_tree_get_plane": (C.c_int, [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp]),
        "orc_tree_get_blocks": (C.c_int, [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp]),
        "orc_search_block": (None, [vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp]),
        "orc_search_block_halfpel": (None, [vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp]),
        "orc_open": (vp, [vp, C.c_size_t, C.POINTER(C.c_int)]),
        "orc_close": (None, [vp]),
        "orc_stream_params": (C.c_int, [vp, C.POINTER(Params)]),
        "orc_set_min_level": (C.c_int, [vp, C.c_int]),
        "orc_decode": (i64, [vp, vp, i64, vp, C.c_int]),
        "orc_decode_brute": (i64, [vp, vp, i64, vp]),
        "orc_decode_full": (C.c_int, [vp, vp, C.c_int]),
        "orc_render": (C.c_int, [vp, vp, C.c_int, C.c_int, C.c_int, vp, C.c_int]),
        "orc_render_dense": (C.c_int, [vp, C.POINTER(Params), vp, C.c_int, C.c_int, C.c_int, vp, C.c_int]),
        "orc_render_lod": (C.c_int, [vp, vp, vp, C.c_int, C.c_int, C.c_int, vp, C.c_int]),
        "orc_lod_level": (C.c_int, [C.POINTER(Params), vp, C.c_float]),
        "orc_ray_setup": (C.c_int, [C.POINTER(Params), vp, C.c_int, C.c_int, vp]),
        "orc_stats_decode": (C.c_int, [vp, vp, i64, C.POINTER(Stats)]),
        "orc_stats_render": (C.c_int, [vp, vp, C.c_int, C.c_int, C.c_int, C.POINTER(Stats)]),
        "orc_psnr": (C.c_double, [vp, vp, i64]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype = res
        f.argtypes = args
    _lib = L
    return L


class OracleError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"oracle: {what} failed with code {code}")
        self.code = code


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def make_params(U, V, Ws, Ht, height, block=4, window=16, tau_ref=0, tau_res=0, policy=POLICY_ADAPTIVE,
                geometry=None, background=(0, 0, 0), seed=0, nthreads=0, chroma=0, subpel=0) -> Params:
    """geometry: dict(uv_origin, uv_step, st_origin, st_step, z_st) or None for the unit slab.
    chroma = 1: Co / Cg planes at half resolution (R18); subpel = 1: half-pel motion compensation
    (R28)."""
    p = Params()
    p.chroma = chroma
    p.subpel = subpel
    p.U, p.V, p.Ws, p.Ht, p.height, p.block, p.window = U, V, Ws, Ht, height, block, window
    p.tau_ref, p.tau_res, p.policy, p.nthreads = tau_ref, tau_res, policy, nthreads
    g = geometry or dict(uv_origin=(0.0, 0.0), uv_step=(1.0, 1.0), st_origin=(0.0, 0.0), st_step=(1.0, 1.0), z_st=1.0)
    for k in ("uv_origin", "uv_step", "st_origin", "st_step"):
        getattr(p, k)[0], getattr(p, k)[1] = float(g[k][0]), float(g[k][1])
    p.z_st = float(g["z_st"])
    for i in range(3):
        p.background[i] = background[i]
    p.seed = seed
    return p


# ------------------------------------------------------------------ colour / BISE
def rgb_to_ycocg(r, g, b):
    y, co, cg = C.c_int(), C.c_int(), C.c_int()
    lib().orc_rgb_to_ycocg(r, g, b, C.byref(y), C.byref(co), C.byref(cg))
    return y.value, co.value, cg.value


def ycocg_to_rgb(y, co, cg):
    r, g, b = C.c_int(), C.c_int(), C.c_int()
    lib().orc_ycocg_to_rgb(y, co, cg, C.byref(r), C.byref(g), C.byref(b))
    return r.value, g.value, b.value


def colour_roundtrip_failures():
    return lib().orc_colour_roundtrip_failures()


def bise_choose(N):
    layout, m = C.c_int32(), C.c_int32()
    lib().orc_bise_choose(N, C.byref(layout), C.byref(m))
    return layout.value, m.value


def bise_nbits(N, count):
    return lib().orc_bise_nbits(N, count)


def bise_encode(values, N) -> np.ndarray:
    v = np.ascontiguousarray(values, dtype=np.uint32)
    nbits = bise_nbits(N, v.size)
    bits = np.zeros(nbits // 8 + 16, dtype=np.uint8)
    rc = lib().orc_bise_encode(_ptr(v), v.size, N, _ptr(bits))
    if rc:
        raise OracleError(rc, "bise_encode")
    return bits


def bise_decode_at(bits, N, i):
    return lib().orc_bise_decode_at(_ptr(bits), N, i)


def bise_decode_seq(bits, N, count) -> np.ndarray:
    out = np.zeros(count, dtype=np.uint32)
    lib().orc_bise_decode_seq(_ptr(bits), N, count, _ptr(out))
    return out


# ------------------------------------------------------------------ encoder
class Tree:
    """The HMLFC tree of one light field (encoder side)."""

    def __init__(self, lf: np.ndarray, params: Params):
        assert lf.dtype == np.uint8 and lf.shape == (params.V, params.U, params.Ht, params.Ws, 3), lf.shape
        self.params = params
        self._lf = np.ascontiguousarray(lf)
        err = C.c_int(0)
        self._h = lib().orc_encode_begin(_ptr(self._lf), C.byref(params), C.byref(err))
        if not self._h:
            raise OracleError(err.value, "encode_begin")

    def close(self):
        if self._h:
            lib().orc_tree_free(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def threshold(self, tau_ref, tau_res, policy=None):
        pol = self.params.policy if policy is None else policy
        rc = lib().orc_tree_threshold(self._h, tau_ref, tau_res, pol)
        if rc:
            raise OracleError(rc, "threshold")
        self.params.tau_ref, self.params.tau_res, self.params.policy = tau_ref, tau_res, pol

    def serialize(self) -> bytes:
        out = C.c_void_p()
        n = lib().orc_tree_serialize(self._h, C.byref(out))
        if n < 0:
            raise OracleError(n, "serialize")
        data = C.string_at(out, n)
        lib().orc_free(out)
        return data

    def reconstruct(self) -> np.ndarray:
        p = self.params
        out = np.empty((p.V, p.U, p.Ht, p.Ws, 3), dtype=np.uint8)
        rc = lib().orc_tree_reconstruct(self._h, _ptr(out))
        if rc:
            raise OracleError(rc, "reconstruct")
        return out

    def level_dims(self, L):
        a, b = C.c_int(), C.c_int()
        rc = lib().orc_tree_level_dims(self._h, L, C.byref(a), C.byref(b))
        if rc:
            raise OracleError(rc, "level_dims")
        return a.value, b.value

    def plane(self, kind, L, pu, pv, c) -> np.ndarray:
        """kind: 'X' | 'srv' | 'stored'."""
        k = {"X": 0, "srv": 1, "stored": 2}[kind]
        sh = 1 if (self.params.chroma and c > 0) else 0   # the channel's own plane size (R18)
        out = np.empty((self.params.Ht >> sh, self.params.Ws >> sh), dtype=np.int16)
        rc = lib().orc_tree_get_plane(self._h, k, L, pu, pv, c, _ptr(out))
        if rc:
            raise OracleError(rc, "get_plane")
        return out

    def blocks(self, L, pu, pv, c) -> np.ndarray:
        """[nby][nbx][6] = mode, dx, dy, sad, E, flags(bit0 res, bit1 pred)."""
        p = self.params
        sh = 1 if (p.chroma and c > 0) else 0
        nbx, nby = (p.Ws >> sh) // p.block, (p.Ht >> sh) // p.block
        out = np.empty((nby, nbx, 6), dtype=np.int32)
        rc = lib().orc_tree_get_blocks(self._h, L, pu, pv, c, _ptr(out))
        if rc:
            raise OracleError(rc, "get_blocks")
        return out


def search_block(P, R, B, W, bx, by):
    P = np.ascontiguousarray(P, dtype=np.int16)
    R = np.ascontiguousarray(R, dtype=np.int16)
    out = np.zeros(4, dtype=np.int32)
    lib().orc_search_block(_ptr(P), _ptr(R), P.shape[1], P.shape[0], B, W, bx, by, _ptr(out))
    return tuple(int(x) for x in out)  # mode, dx, dy, sad


def search_block_halfpel(P, R, B, W, bx, by):
    """The search on the half-pel grid (R28): (mode, dx2, dy2, sad), offsets in half pixels."""
    P = np.ascontiguousarray(P, dtype=np.int16)
    R = np.ascontiguousarray(R, dtype=np.int16)
    out = np.zeros(4, dtype=np.int32)
    lib().orc_search_block_halfpel(_ptr(P), _ptr(R), P.shape[1], P.shape[0], B, W, bx, by, _ptr(out))
    return tuple(int(x) for x in out)


def psnr(a, b) -> float:
    a = np.ascontiguousarray(a, dtype=np.uint8)
    b = np.ascontiguousarray(b, dtype=np.uint8)
    assert a.shape == b.shape
    return lib().orc_psnr(_ptr(a), _ptr(b), a.size)


# ------------------------------------------------------------------ decoder / renderer
class Stream:
    """A parsed compressed stream (decoder side)."""

    def __init__(self, data: bytes):
        err = C.c_int(0)
        buf = np.frombuffer(data, dtype=np.uint8)
        self._h = lib().orc_open(_ptr(buf), buf.size, C.byref(err))
        if not self._h:
            raise OracleError(err.value, "open")
        self.params = Params()
        lib().orc_stream_params(self._h, C.byref(self.params))
        self.nbytes = len(data)

    def close(self):
        if self._h:
            lib().orc_close(self._h)
            self._h = None

    def __del__(self):
        self.close()

    def set_min_level(self, min_level):
        """Progressive decoding: sum only the levels >= min_level (0 = full quality, height = top RKV only)."""
        rc = lib().orc_set_min_level(self._h, min_level)
        if rc:
            raise OracleError(rc, "set_min_level")

    def decode(self, coords, nthreads=0, return_oob=False):
        c = np.ascontiguousarray(coords, dtype=np.int32).reshape(-1, 4)
        out = np.empty((c.shape[0], 3), dtype=np.uint8)
        oob = lib().orc_decode(self._h, _ptr(c), c.shape[0], _ptr(out), nthreads)
        if oob < 0:
            raise OracleError(oob, "decode")
        return (out, oob) if return_oob else out

    def decode_brute(self, coords):
        c = np.ascontiguousarray(coords, dtype=np.int32).reshape(-1, 4)
        out = np.empty((c.shape[0], 3), dtype=np.uint8)
        oob = lib().orc_decode_brute(self._h, _ptr(c), c.shape[0], _ptr(out))
        if oob < 0:
            raise OracleError(oob, "decode_brute")
        return out

    def decode_full(self, nthreads=0):
        p = self.params
        out = np.empty((p.V, p.U, p.Ht, p.Ws, 3), dtype=np.uint8)
        rc = lib().orc_decode_full(self._h, _ptr(out), nthreads)
        if rc:
            raise OracleError(rc, "decode_full")
        return out

    def render(self, cams, W, H, nthreads=0):
        cams = np.ascontiguousarray(cams, dtype=np.float32).reshape(-1, 16)
        out = np.empty((cams.shape[0], H, W, 3), dtype=np.uint8)
        rc = lib().orc_render(self._h, _ptr(cams), cams.shape[0], W, H, _ptr(out), nthreads)
        if rc:
            raise OracleError(rc, "render")
        return out

    def render_lod(self, cams, levels, W, H, nthreads=0):
        """Per-view level of detail (R27): view k is rendered with the walk stopped above levels[k]."""
        cams = np.ascontiguousarray(cams, dtype=np.float32).reshape(-1, 16)
        levels = np.ascontiguousarray(levels, dtype=np.int32)
        assert levels.shape == (cams.shape[0],)
        out = np.empty((cams.shape[0], H, W, 3), dtype=np.uint8)
        rc = lib().orc_render_lod(self._h, _ptr(cams), _ptr(levels), cams.shape[0], W, H, _ptr(out), nthreads)
        if rc:
            raise OracleError(rc, "render_lod")
        return out

    def lod_levels(self, cams, d0):
        """floor(log2(|z_st - eye.z| / d0)) clamped to [0, height], per camera."""
        cams = np.ascontiguousarray(cams, dtype=np.float32).reshape(-1, 16)
        p = self.params
        return np.array([lib().orc_lod_level(C.byref(p), _ptr(cams[k]), C.c_float(d0)) for k in range(cams.shape[0])], dtype=np.int32)

    def stats_decode(self, coords):
        c = np.ascontiguousarray(coords, dtype=np.int32).reshape(-1, 4)
        st = Stats()
        rc = lib().orc_stats_decode(self._h, _ptr(c), c.shape[0], C.byref(st))
        if rc:
            raise OracleError(rc, "stats_decode")
        return st.as_dict()

    def stats_render(self, cams, W, H):
        cams = np.ascontiguousarray(cams, dtype=np.float32).reshape(-1, 16)
        st = Stats()
        rc = lib().orc_stats_render(self._h, _ptr(cams), cams.shape[0], W, H, C.byref(st))
        if rc:
            raise OracleError(rc, "stats_render")
        return st.as_dict()


def render_dense(lf, params, cams, W, H, nthreads=0):
    lf = np.ascontiguousarray(lf, dtype=np.uint8)
    cams = np.ascontiguousarray(cams, dtype=np.float32).reshape(-1, 16)
    out = np.empty((cams.shape[0], H, W, 3), dtype=np.uint8)
    rc = lib().orc_render_dense(_ptr(lf), C.byref(params), _ptr(cams), cams.shape[0], W, H, _ptr(out), nthreads)
    if rc:
        raise OracleError(rc, "render_dense")
    return out


def ray_setup(params, cam, W, H):
    cam = np.ascontiguousarray(cam, dtype=np.float32).reshape(16)
    out = np.empty((H, W, 5), dtype=np.float32)
    rc = lib().orc_ray_setup(C.byref(params), _ptr(cam), W, H, _ptr(out))
    if rc:
        raise OracleError(rc, "ray_setup")
    return out


def encode(lf, params, target_psnr=None, tol=0.25, max_iter=12):
    """Encode a light field.  If target_psnr is given, bisect tau_res (tau_ref = tau_res // 2, reading
    R24) until the P1 reconstruction's PSNR is within tol of the target.
    Returns (stream_bytes, info dict, tree)."""
    tree = Tree(lf, params)
    info = {}
    if target_psnr is not None:
        lo, hi = 0, 4096
        best = None
        for _ in range(max_iter):
            mid = (lo + hi) // 2
            tree.threshold(mid // 2, mid)
            q = psnr(tree.reconstruct(), lf)
            if best is None or abs(q - target_psnr) < abs(best[1] - target_psnr):
                best = (mid, q)
            if abs(q - target_psnr) <= tol or hi - lo <= 1:
                break
            if q > target_psnr:
                lo = mid
            else:
                hi = mid
        tree.threshold(best[0] // 2, best[0])
    data = tree.serialize()
    rec = tree.reconstruct()
    info["psnr"] = psnr(rec, lf)
    info["tau_res"], info["tau_ref"] = tree.params.tau_res, tree.params.tau_ref
    info["bpp"] = 8.0 * len(data) / (params.U * params.V * params.Ws * params.Ht)
    info["stream_bytes"] = len(data)
    return data, info, tree
