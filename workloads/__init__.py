"""Seeded synthetic workloads: light fields, camera paths, coordinate lists.

This module serves BOTH the oracle (tests, baselines) and the CUDA path (bench, tests) and
holds none of HMLFC's arithmetic: it only makes inputs.  Recipe: DESIGN.md "Input recipe"
(after SURVEY.md 8(d) D1-D4).  The five configurations are BASELINE.json's `configs`.

World units = camera spacing b = 1.  Camera (iu,iv) sits at (iu, iv, 0); pixel (is,it) of the
common image plane sits at (st_origin + (is,it)/16, z_st): pixel pitch p = b/16, so a
fronto-parallel plane at depth z has per-view-step disparity delta = 16 (1 - z_st / z) pixels.
"""
import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(HERE, "libworkloads.so")
BASE_SEED = 190209396
PITCH = 1.0 / 16.0  # p / b


@dataclass(frozen=True)
class Config:
    name: str
    U: int
    V: int
    Ws: int
    Ht: int
    height: int
    n_planes: int
    n_spheres: int
    delta_max: float
    target_psnr: float | None   # None: use tau_res as given
    tau_res: int
    out_w: int
    out_h: int
    n_views: int                # views per render batch
    n_decode: int               # coordinates of the decode workload
    noise_sigma: float = 0.0
    deltas: tuple = ()          # explicit plane disparities (cfg1)
    seed: int = BASE_SEED
    block: int = 4
    window: int = 16


CONFIGS = {
    # BASELINE.json configs[0..4]
    "cfg1": Config("cfg1", 8, 8, 64, 64, 2, 3, 0, 3.0, None, 0, 64, 64, 1, 8 * 8 * 64 * 64, noise_sigma=2.0,
                   deltas=(0.0, 1.5, 3.0), seed=BASE_SEED + 1),
    "cfg1_lossy": Config("cfg1_lossy", 8, 8, 64, 64, 2, 3, 0, 3.0, None, 40, 64, 64, 1, 8 * 8 * 64 * 64,
                         noise_sigma=2.0, deltas=(0.0, 1.5, 3.0), seed=BASE_SEED + 1),
    "cfg2": Config("cfg2", 16, 16, 256, 256, 3, 5, 2, 4.0, 40.0, 0, 512, 512, 64, 10 ** 7, seed=BASE_SEED + 2),
    "cfg3": Config("cfg3", 17, 17, 512, 512, 3, 8, 4, 6.0, 45.0, 0, 512, 512, 16, 10 ** 7, seed=BASE_SEED + 3),
    "cfg4": Config("cfg4", 32, 32, 512, 512, 4, 12, 8, 8.0, 40.0, 0, 1024, 1024, 16, 10 ** 8, seed=BASE_SEED + 4),
    "cfg5": Config("cfg5", 64, 64, 640, 640, 4, 20, 16, 10.0, 40.0, 0, 2048, 2048, 8, 10 ** 8, seed=BASE_SEED + 5),
    # reduced shapes for parity tests the oracle finishes in seconds (same recipe, same structure)
    "mini2": Config("mini2", 8, 8, 96, 80, 3, 5, 2, 4.0, None, 48, 200, 136, 3, 50_000, seed=BASE_SEED + 12),
    "mini3": Config("mini3", 5, 5, 64, 48, 3, 4, 2, 6.0, None, 30, 100, 76, 2, 30_000, seed=BASE_SEED + 13),
    "mini4": Config("mini4", 16, 16, 64, 64, 4, 6, 3, 8.0, None, 48, 160, 120, 2, 50_000, seed=BASE_SEED + 14),
    # other block sizes / search windows (the paper's Table 2 sweeps B = 2, 4, 8)
    "mini_b2": Config("mini_b2", 4, 4, 48, 40, 2, 4, 1, 3.0, None, 12, 90, 70, 2, 20_000, seed=BASE_SEED + 15, block=2, window=5),
    "mini_b8": Config("mini_b8", 5, 4, 64, 48, 2, 4, 2, 4.0, None, 160, 120, 88, 2, 20_000, seed=BASE_SEED + 16, block=8, window=8),
    # the limits of the stream format: tree height 8 (levels 6x5 -> 3x3 -> 2x2 -> 1x1 x 5: a cluster of one
    # plane has SRV = 0 at every level above) and search window 64 (129 x 129 offsets, wider than the image)
    "mini_h8": Config("mini_h8", 6, 5, 32, 24, 8, 3, 1, 3.0, None, 24, 72, 56, 2, 20_000, seed=BASE_SEED + 17, window=4),
    "mini_w64": Config("mini_w64", 3, 2, 24, 16, 2, 3, 1, 3.0, None, 20, 56, 40, 2, 10_000, seed=BASE_SEED + 18, window=64),
    # search windows whose motion-record alphabet N = 2 (2W+1)^2 takes the trit layout with m = 11 / 12 / 13 / 13: BISE groups of
    # 63 / 68 / 73 bits, longer than any payload group (the record fields end beyond a 96-bit window)
    "mini_w25": Config("mini_w25", 4, 4, 48, 32, 2, 3, 1, 3.0, None, 16, 72, 48, 2, 10_000, seed=BASE_SEED + 19, window=25),
    "mini_w37": Config("mini_w37", 4, 4, 48, 32, 2, 3, 1, 3.0, None, 16, 72, 48, 2, 10_000, seed=BASE_SEED + 20, window=37),
    "mini_w51": Config("mini_w51", 4, 4, 48, 32, 2, 3, 1, 3.0, None, 16, 72, 48, 2, 10_000, seed=BASE_SEED + 21, window=51),
    "mini_w54": Config("mini_w54", 4, 4, 48, 32, 2, 3, 1, 3.0, None, 16, 72, 48, 2, 10_000, seed=BASE_SEED + 23, window=54),
    # paper-regime sparsity: adjacent views < 1 px apart, as in the Stanford archive
    "cfg2_sparse": Config("cfg2_sparse", 16, 16, 256, 256, 3, 5, 2, 1.0, 40.0, 0, 512, 512, 64, 10 ** 7,
                          seed=BASE_SEED + 22),
}


def geometry(cfg: Config) -> dict:
    """Light-slab geometry of a configuration (float32-representable values)."""
    z_st = 0.5 * (cfg.U - 1)
    cx, cy = 0.5 * (cfg.U - 1), 0.5 * (cfg.V - 1)
    return dict(
        uv_origin=(0.0, 0.0), uv_step=(1.0, 1.0),
        st_origin=(cx - 0.5 * (cfg.Ws - 1) * PITCH, cy - 0.5 * (cfg.Ht - 1) * PITCH),
        st_step=(PITCH, PITCH), z_st=z_st,
    )


# ------------------------------------------------------------------ light-field generator (C)
class _Scene(C.Structure):
    _fields_ = [("U", C.c_int32), ("V", C.c_int32), ("Ws", C.c_int32), ("Ht", C.c_int32),
                ("uv_origin", C.c_double * 2), ("uv_step", C.c_double * 2), ("st_origin", C.c_double * 2),
                ("st_step", C.c_double * 2), ("z_st", C.c_double), ("n_planes", C.c_int32), ("n_spheres", C.c_int32),
                ("noise_sigma", C.c_double), ("seed", C.c_uint64), ("light", C.c_double * 3),
                ("base_cell_px", C.c_double)]


class _Plane(C.Structure):
    _fields_ = [("z", C.c_double), ("x0", C.c_double), ("x1", C.c_double), ("y0", C.c_double), ("y1", C.c_double),
                ("base", C.c_double * 3), ("tex", C.c_uint64)]


class _Sphere(C.Structure):
    _fields_ = [("c", C.c_double * 3), ("r", C.c_double), ("base", C.c_double * 3), ("tex", C.c_uint64)]


def build_lib(force=False) -> str:
    src = os.path.join(HERE, "lfgen.c")
    if force or not os.path.exists(_LIB) or os.path.getmtime(src) > os.path.getmtime(_LIB):
        subprocess.run(["gcc", "-std=c11", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB + ".tmp",
                        src, "-lm"], check=True)
        os.replace(_LIB + ".tmp", _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_lib())
        _lib.wl_generate_lf.restype = C.c_int
        _lib.wl_generate_lf.argtypes = [C.POINTER(_Scene), C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
    return _lib


def scene(cfg: Config):
    """Seeded scene description: (planes, spheres) as plain dict lists."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    g = geometry(cfg)
    z_st = g["z_st"]
    ccx, ccy = 0.5 * (cfg.U - 1), 0.5 * (cfg.V - 1)
    fw, fh = (cfg.Ws - 1) * PITCH, (cfg.Ht - 1) * PITCH  # st rectangle size (world units)
    if cfg.deltas:
        deltas = np.array(cfg.deltas, dtype=np.float64)
    else:
        deltas = rng.uniform(-cfg.delta_max, cfg.delta_max, cfg.n_planes)
    order = np.argsort(-deltas)  # farthest (largest delta) first
    planes = []
    for rank, k in enumerate(order):
        d = float(deltas[k])
        z = z_st / (1.0 - d * PITCH)
        base = rng.uniform(0.0, 1.0, 3)
        tex = int(rng.integers(1, 2 ** 62))
        if rank == 0:
            x0, x1, y0, y1 = -1e30, 1e30, -1e30, 1e30  # the farthest plane fills the frame
        else:
            wx, wy = rng.uniform(0.4, 0.7, 2)
            ox, oy = rng.uniform(0.0, 1.0 - wx), rng.uniform(0.0, 1.0 - wy)
            # rectangle on the st plane (as seen from the central camera), pushed to depth z
            sx0, sx1 = g["st_origin"][0] + ox * fw, g["st_origin"][0] + (ox + wx) * fw
            sy0, sy1 = g["st_origin"][1] + oy * fh, g["st_origin"][1] + (oy + wy) * fh
            x0, x1 = ccx + (sx0 - ccx) * z / z_st, ccx + (sx1 - ccx) * z / z_st
            y0, y1 = ccy + (sy0 - ccy) * z / z_st, ccy + (sy1 - ccy) * z / z_st
        planes.append(dict(z=z, x0=x0, x1=x1, y0=y0, y1=y1, base=base, tex=tex, delta=d))
    spheres = []
    for _ in range(cfg.n_spheres):
        d = float(rng.uniform(-cfg.delta_max, cfg.delta_max))
        z = z_st / (1.0 - d * PITCH)
        px, py = rng.uniform(0.15, 0.85, 2)
        sx, sy = g["st_origin"][0] + px * fw, g["st_origin"][1] + py * fh
        r_px = rng.uniform(0.05, 0.15) * cfg.Ws
        spheres.append(dict(c=(ccx + (sx - ccx) * z / z_st, ccy + (sy - ccy) * z / z_st, z), r=r_px * PITCH * z / z_st,
                            base=rng.uniform(0.0, 1.0, 3), tex=int(rng.integers(1, 2 ** 62)), delta=d))
    return planes, spheres


def light_field(cfg: Config, nthreads=0) -> np.ndarray:
    """RGB8 light field [V][U][Ht][Ws][3] of a configuration."""
    planes, spheres = scene(cfg)
    g = geometry(cfg)
    sc = _Scene()
    sc.U, sc.V, sc.Ws, sc.Ht = cfg.U, cfg.V, cfg.Ws, cfg.Ht
    for k in ("uv_origin", "uv_step", "st_origin", "st_step"):
        getattr(sc, k)[0], getattr(sc, k)[1] = g[k]
    sc.z_st = g["z_st"]
    sc.n_planes, sc.n_spheres = len(planes), len(spheres)
    sc.noise_sigma, sc.seed = cfg.noise_sigma, cfg.seed
    l = np.array([-0.4, -0.5, -0.77])
    l /= np.linalg.norm(l)
    sc.light[0], sc.light[1], sc.light[2] = l
    sc.base_cell_px = cfg.Ws / 4.0
    P = (_Plane * max(1, len(planes)))()
    for i, p in enumerate(planes):
        P[i].z, P[i].x0, P[i].x1, P[i].y0, P[i].y1, P[i].tex = p["z"], p["x0"], p["x1"], p["y0"], p["y1"], p["tex"]
        P[i].base[0], P[i].base[1], P[i].base[2] = p["base"]
    S = (_Sphere * max(1, len(spheres)))()
    for i, s in enumerate(spheres):
        S[i].c[0], S[i].c[1], S[i].c[2] = s["c"]
        S[i].r, S[i].tex = s["r"], s["tex"]
        S[i].base[0], S[i].base[1], S[i].base[2] = s["base"]
    lf = np.empty((cfg.V, cfg.U, cfg.Ht, cfg.Ws, 3), dtype=np.uint8)
    rc = _load().wl_generate_lf(C.byref(sc), P, S, lf.ctypes.data_as(C.c_void_p), nthreads)
    if rc:
        raise RuntimeError(f"wl_generate_lf failed: {rc}")
    return lf


# ------------------------------------------------------------------ cameras
def _camera(eye, look, tan_half_x, tan_half_y) -> np.ndarray:
    eye, look = np.asarray(eye, np.float64), np.asarray(look, np.float64)
    fwd = look - eye
    fwd /= np.linalg.norm(fwd)
    right = np.cross(np.array([0.0, 1.0, 0.0]), fwd)
    right /= np.linalg.norm(right)
    down = np.cross(fwd, right)
    cam = np.zeros(16, dtype=np.float32)
    cam[0:3], cam[3:6], cam[6:9], cam[9:12] = eye, right, down, fwd
    cam[12], cam[13] = tan_half_x, tan_half_y
    return cam


def camera_path(cfg: Config, n_views=None, out_w=None, out_h=None, seed_offset=0, phase=None, on_plane=False) -> np.ndarray:
    """n_views cameras on the seeded circular path of DESIGN.md "Input recipe":
    eye on a circle of radius 0.25 (U-1) around the uv-rectangle centre at z = -0.25 (U-1), looking at the
    st-rectangle centre; the frustum covers ~80% of the st rectangle.  Returns float32 [n_views][16].
    on_plane: the "grid-aligned" batch of SURVEY 8(d) D4 -- the same circle ON the camera plane (z = 0), so every ray of a
    view meets the uv plane at the eye and a whole view blends exactly the 4 views around it (best case for sharing)."""
    n_views = cfg.n_views if n_views is None else n_views
    out_w, out_h = out_w or cfg.out_w, out_h or cfg.out_h
    rng = np.random.Generator(np.random.PCG64(cfg.seed + 1000 + seed_offset))
    g = geometry(cfg)
    ccx, ccy = 0.5 * (cfg.U - 1), 0.5 * (cfg.V - 1)
    rad, ze = 0.25 * (cfg.U - 1), (0.0 if on_plane else -0.25 * (cfg.U - 1))
    look = np.array([g["st_origin"][0] + 0.5 * (cfg.Ws - 1) * PITCH, g["st_origin"][1] + 0.5 * (cfg.Ht - 1) * PITCH, g["z_st"]])
    start = rng.uniform(0.0, 2.0 * np.pi) if phase is None else phase
    cams = np.zeros((n_views, 16), dtype=np.float32)
    for k in range(n_views):
        a = start + 2.0 * np.pi * k / max(1, n_views)
        if n_views == 1:  # cfg1: seeded eye inside the disc, seeded look-at in the central half
            r = rad * np.sqrt(rng.uniform())
            eye = np.array([ccx + r * np.cos(a), ccy + r * np.sin(a), ze])
            lk = look + np.array([rng.uniform(-0.25, 0.25) * (cfg.Ws - 1) * PITCH, rng.uniform(-0.25, 0.25) * (cfg.Ht - 1) * PITCH, 0.0])
        else:
            eye = np.array([ccx + rad * np.cos(a), ccy + rad * np.sin(a), ze])
            lk = look
        d = np.linalg.norm(lk - eye)
        thx = 0.4 * (cfg.Ws - 1) * PITCH / d
        cams[k] = _camera(eye, lk, thx, thx * out_h / out_w)
    return cams


def grid_camera(cfg: Config, iu: int, iv: int) -> np.ndarray:
    """Camera at grid viewpoint (iu,iv) whose Ws x Ht frustum reproduces that view exactly
    (SURVEY.md 8(c) C7 "self-reprojection")."""
    g = geometry(cfg)
    z = g["z_st"]
    ex, ey = g["uv_origin"][0] + iu * g["uv_step"][0], g["uv_origin"][1] + iv * g["uv_step"][1]
    cam = np.zeros(16, dtype=np.float32)
    cam[0:3] = (ex, ey, 0.0)
    cam[3:6] = (1.0, 0.0, 0.0)
    cam[6:9] = (0.0, 1.0, 0.0)
    cam[9:12] = ((g["st_origin"][0] + (cfg.Ws / 2 - 0.5) * g["st_step"][0] - ex) / z,
                 (g["st_origin"][1] + (cfg.Ht / 2 - 0.5) * g["st_step"][1] - ey) / z, 1.0)
    cam[12] = cfg.Ws * g["st_step"][0] / (2.0 * z)
    cam[13] = cfg.Ht * g["st_step"][1] / (2.0 * z)
    return cam


# ------------------------------------------------------------------ coordinates
def random_coords(cfg: Config, n=None, seed_offset=0) -> np.ndarray:
    """n seeded uniformly random LF pixel coordinates, int32 [n][4] = (u, v, s, t)."""
    n = cfg.n_decode if n is None else n
    rng = np.random.Generator(np.random.PCG64(cfg.seed + 2000 + seed_offset))
    out = np.empty((n, 4), dtype=np.int32)
    out[:, 0] = rng.integers(0, cfg.U, n, dtype=np.int32)
    out[:, 1] = rng.integers(0, cfg.V, n, dtype=np.int32)
    out[:, 2] = rng.integers(0, cfg.Ws, n, dtype=np.int32)
    out[:, 3] = rng.integers(0, cfg.Ht, n, dtype=np.int32)
    return out


def srv_like_planes(cfg: Config, n_planes: int, seed_offset=0) -> np.ndarray:
    """n_planes signed int16 images [n][Ht][Ws] with the statistics of SRV images (differences of neighbouring views:
    zero-mean, a few tens in magnitude, locally coherent, each plane a shifted and sometimes sign-inverted copy of a
    common signal plus noise).  Input of the encoder-side search timing; holds no HMLFC arithmetic."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed + 3000 + seed_offset))
    pad = 16
    base = rng.normal(0.0, 40.0, (cfg.Ht + 2 * pad, cfg.Ws + 2 * pad))
    for _ in range(2):  # a little spatial coherence
        base = 0.25 * (base + np.roll(base, 1, 0) + np.roll(base, 1, 1) + np.roll(base, (1, 1), (0, 1))) * 1.6
    out = np.empty((n_planes, cfg.Ht, cfg.Ws), dtype=np.int16)
    for k in range(n_planes):
        dx, dy = rng.integers(-pad, pad + 1, 2)
        sign = -1.0 if rng.uniform() < 0.45 else 1.0
        img = sign * base[pad + dy:pad + dy + cfg.Ht, pad + dx:pad + dx + cfg.Ws] + rng.normal(0.0, 3.0, (cfg.Ht, cfg.Ws))
        out[k] = np.clip(np.rint(img), -510, 510).astype(np.int16)
    return out


def all_coords(cfg: Config) -> np.ndarray:
    """Every LF pixel once, in [V][U][Ht][Ws] order (cfg1's exhaustive decode)."""
    v, u, t, s = np.meshgrid(np.arange(cfg.V), np.arange(cfg.U), np.arange(cfg.Ht), np.arange(cfg.Ws), indexing="ij")
    return np.stack([u, v, s, t], axis=-1).reshape(-1, 4).astype(np.int32)


def shard(n_items: int, rank: int, world: int):
    """Contiguous [lo, hi) share of n_items for `rank` of `world`."""
    base, rem = divmod(n_items, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
