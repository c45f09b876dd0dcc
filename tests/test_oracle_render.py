"""Pins for the oracle's two-plane renderer
and for the synthetic workload generator."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl


def _cfg(U, V, Ws, Ht, h=2, **kw):
    return wl.Config("t", U, V, Ws, Ht, h, 1, 0, 0.0, None, 0, Ws, Ht, 1, 0, **kw)


def _stream(lf, cfg, tau=0, W=4, bg=(0, 0, 0)):
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, 4, W, tau // 2, tau, geometry=wl.geometry(cfg), background=bg)
    data, info, tree = orc.encode(lf, p)
    return orc.Stream(data), p


def _free_camera(cfg, rng):
    """A rotated, off-plane camera whose rays mostly hit the slab."""
    g = wl.geometry(cfg)
    c = np.array([0.5 * (cfg.U - 1), 0.5 * (cfg.V - 1)])
    eye = np.array([c[0] + rng.uniform(-1, 1), c[1] + rng.uniform(-1, 1), -rng.uniform(0.5, 2.0)])
    look = np.array([c[0] + rng.uniform(-0.5, 0.5), c[1] + rng.uniform(-0.5, 0.5), g["z_st"]])
    d = np.linalg.norm(look - eye)
    return wl._camera(eye, look, 0.3 * (cfg.Ws - 1) * wl.PITCH / d, 0.3 * (cfg.Ht - 1) * wl.PITCH / d)


# ---------------------------------------------------------------- ray set-up
def test_ray_through_plane_centres_and_parallel_miss():
    cfg = _cfg(8, 8, 64, 64)
    g = wl.geometry(cfg)
    p = orc.make_params(8, 8, 64, 64, 2, geometry=g)
    # ray orthogonal through the plane centres -> (centre, centre)
    cam = np.zeros(16, np.float32)
    cam[0:3] = (3.5, 3.5, -2.0)
    cam[3:6], cam[6:9], cam[9:12] = (1, 0, 0), (0, 1, 0), (0, 0, 1)
    cam[12] = cam[13] = 1e-6
    r = orc.ray_setup(p, cam, 1, 1)[0, 0]
    assert r[4] == 1.0 and np.allclose(r[:4], [3.5, 3.5, 31.5, 31.5], atol=1e-3)
    # ray parallel to the planes -> miss
    cam[9:12] = (1, 0, 0)
    cam[3:6] = (0, 0, 1)
    cam[12] = cam[13] = 0.0
    assert orc.ray_setup(p, cam, 1, 1)[0, 0, 4] == 0.0


def test_ray_setup_matches_float64_line_plane_intersection():
    # independent analytic oracle (float64), tolerance = fp32 rounding
    rng = np.random.default_rng(0)
    cfg = _cfg(8, 8, 64, 48)
    g = wl.geometry(cfg)
    p = orc.make_params(8, 8, 64, 48, 2, geometry=g)
    cam = _free_camera(cfg, rng)
    W, H = 40, 30
    rays = orc.ray_setup(p, cam, W, H)
    eye, right, down, fwd = (cam[i:i + 3].astype(np.float64) for i in (0, 3, 6, 9))
    n_hit = 0
    for j in range(H):
        for i in range(W):
            px = (2 * (i + 0.5) / W - 1) * float(cam[12])
            py = (2 * (j + 0.5) / H - 1) * float(cam[13])
            D = fwd + px * right + py * down
            Puv = eye + (0 - eye[2]) / D[2] * D
            Pst = eye + (g["z_st"] - eye[2]) / D[2] * D
            u, v = Puv[0], Puv[1]
            s = (Pst[0] - g["st_origin"][0]) / wl.PITCH
            t = (Pst[1] - g["st_origin"][1]) / wl.PITCH
            inside = 0 <= u <= 7 and 0 <= v <= 7 and 0 <= s <= 63 and 0 <= t <= 47
            margin = min(u, 7 - u, v, 7 - v, s, 63 - s, t, 47 - t)
            if abs(margin) > 1e-3:
                assert rays[j, i, 4] == (1.0 if inside else 0.0)
            if rays[j, i, 4] == 1.0:
                n_hit += 1
                assert np.allclose(rays[j, i, :4], [u, v, s, t], atol=2e-3)
    assert n_hit > 200


# ---------------------------------------------------------------- sampling
def test_grid_camera_reproduces_the_view_bit_exactly():
    # SPEC.md:527/536 + SURVEY C7: camera at a grid viewpoint with the matched off-axis frustum
    rng = np.random.default_rng(1)
    cfg = _cfg(8, 8, 64, 64)
    lf = rng.integers(0, 256, (8, 8, 64, 64, 3)).astype(np.uint8)
    p = orc.make_params(8, 8, 64, 64, 2, geometry=wl.geometry(cfg))
    for iu, iv in [(0, 0), (3, 5), (7, 7), (6, 1)]:
        img = orc.render_dense(lf, p, wl.grid_camera(cfg, iu, iv), 64, 64)[0]
        assert np.array_equal(img, lf[iv, iu])


def test_grid_camera_non_square():
    rng = np.random.default_rng(2)
    cfg = _cfg(4, 6, 48, 32)
    lf = rng.integers(0, 256, (6, 4, 32, 48, 3)).astype(np.uint8)
    p = orc.make_params(4, 6, 48, 32, 2, geometry=wl.geometry(cfg))
    img = orc.render_dense(lf, p, wl.grid_camera(cfg, 2, 4), 48, 32)[0]
    assert np.array_equal(img, lf[4, 2])


def test_identical_views_make_output_independent_of_uv():
    # with identical views only (s,t) matters -> bilinear sample of the image
    rng = np.random.default_rng(3)
    cfg = _cfg(4, 4, 32, 32)
    img = rng.integers(0, 256, (32, 32, 3)).astype(np.uint8)
    lf = np.broadcast_to(img, (4, 4, 32, 32, 3)).copy()
    p = orc.make_params(4, 4, 32, 32, 2, geometry=wl.geometry(cfg))
    cam = _free_camera(cfg, rng)
    out = orc.render_dense(lf, p, cam, 24, 24)[0]
    rays = orc.ray_setup(p, cam, 24, 24)
    for j in range(24):
        for i in range(24):
            u, v, s, t, hit = rays[j, i]
            if not hit:
                assert not out[j, i].any()
                continue
            s0, t0 = int(np.floor(s)), int(np.floor(t))
            s1, t1 = min(s0 + 1, 31), min(t0 + 1, 31)
            fs, ft = float(s) - s0, float(t) - t0
            val = ((1 - fs) * (1 - ft) * img[t0, s0].astype(float) + fs * (1 - ft) * img[t0, s1] +
                   (1 - fs) * ft * img[t1, s0] + fs * ft * img[t1, s1])
            assert np.all(np.abs(out[j, i] - val) <= 0.5 + 1e-3)


def test_affine_light_field_closed_form():
    # quadrilinear interpolation reproduces affine functions: out = round(a u + b v + c s + d t + e) +- rounding
    cfg = _cfg(8, 8, 64, 64)
    v, u, t, s = np.meshgrid(np.arange(8), np.arange(8), np.arange(64), np.arange(64), indexing="ij")
    coef = [(3, 2, 1, 2, 10), (1, 4, 2, 1, 5), (2, 2, 1, 1, 60)]
    lf = np.stack([a * u + b * v + c * s + d * t + e for a, b, c, d, e in coef], -1).astype(np.uint8)
    stream, p = _stream(lf, cfg)
    rng = np.random.default_rng(4)
    cam = _free_camera(cfg, rng)
    out = stream.render(cam, 48, 40)[0]
    rays = orc.ray_setup(p, cam, 48, 40)
    hit = rays[..., 4] == 1.0
    assert hit.mean() > 0.5
    for ch, (a, b, c, d, e) in enumerate(coef):
        exact = a * rays[..., 0].astype(np.float64) + b * rays[..., 1] + c * rays[..., 2] + d * rays[..., 3] + e
        assert np.max(np.abs(out[..., ch][hit] - exact[hit])) <= 0.5 + 1e-3
    assert not out[~hit].any()


def test_render_from_stream_equals_render_from_decoded_lf(enc):
    # SPEC.md:541
    cfg, lf, data, info, s = enc("mini2")
    cams = wl.camera_path(cfg)
    a = s.render(cams, cfg.out_w, cfg.out_h)
    b = orc.render_dense(info["p1"], s.params, cams, cfg.out_w, cfg.out_h)
    assert np.array_equal(a, b)
    assert np.array_equal(a, s.render(cams, cfg.out_w, cfg.out_h, nthreads=1))  # thread-count invariant


def test_background_on_miss():
    cfg = _cfg(4, 4, 16, 16)
    lf = np.full((4, 4, 16, 16, 3), 99, np.uint8)
    stream, p = _stream(lf, cfg, bg=(7, 8, 9))
    cam = wl.grid_camera(cfg, 1, 1).copy()
    cam[12] *= 3.0  # three times the frustum: the border misses the st rectangle
    out = stream.render(cam, 48, 16)[0]
    assert np.array_equal(out[0, 0], [7, 8, 9]) and np.array_equal(out[8, 24], [99, 99, 99])


# ---------------------------------------------------------------- workloads
def test_light_field_generator_is_deterministic_and_has_the_stated_disparities():
    cfg = wl.Config("d", 4, 1, 128, 32, 1, 1, 0, 3.0, None, 0, 8, 8, 1, 0, deltas=(2.0,), seed=5)
    a, b = wl.light_field(cfg), wl.light_field(cfg, nthreads=1)
    assert np.array_equal(a, b)
    # one plane at disparity delta = 2 px per view step: view u+1 is view u shifted by 2 px (sign: content moves to -s)
    x = a[0, 0, :, 8:-8].astype(int)
    errs = [np.abs(a[0, 1, :, 8 + d:a.shape[3] - 8 + d].astype(int) - x).mean() for d in range(-4, 5)]
    assert abs(int(np.argmin(errs)) - 4) == 2 and min(errs) < 0.6


def test_zero_disparity_plane_gives_identical_views():
    cfg = wl.Config("d", 3, 3, 32, 32, 1, 1, 0, 0.0, None, 0, 8, 8, 1, 0, deltas=(0.0,), seed=6)
    lf = wl.light_field(cfg)
    assert all(np.array_equal(lf[0, 0], lf[v, u]) for v in range(3) for u in range(3))


def test_cameras_coords_and_sharding_are_seeded():
    cfg = wl.CONFIGS["cfg2"]
    assert np.array_equal(wl.camera_path(cfg), wl.camera_path(cfg))
    c = wl.random_coords(cfg, 1000)
    assert np.array_equal(c, wl.random_coords(cfg, 1000)) and c.dtype == np.int32
    assert c[:, 0].max() < cfg.U and c[:, 3].max() < cfg.Ht and c.min() >= 0
    spans = [wl.shard(64, r, 3) for r in range(3)]
    assert spans == [(0, 22), (22, 43), (43, 64)]
    assert wl.all_coords(wl.CONFIGS["cfg1"]).shape == (262144, 4)


def test_per_view_level_of_detail_is_the_progressive_decoder_view_by_view():
    # R27: view k rendered at level levels[k] = the R26 decoder at that level on that view alone (R26 is pinned by the hierarchy itself:
    # level L of a lossless stream is the cluster key view X_L); the distance rule is floor(log2(d / d0)) clamped to [0, h]
    import workloads as wl

    cfg = wl.CONFIGS["mini3"]
    lf = wl.light_field(cfg)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, 10, 20, geometry=wl.geometry(cfg))
    t = orc.Tree(lf, p)
    s = orc.Stream(t.serialize())
    t.close()
    cams = wl.camera_path(cfg)
    n = cams.shape[0]
    levels = np.arange(n, dtype=np.int32) % (cfg.height + 1)
    got = s.render_lod(cams, levels, 40, 28)
    for k in range(n):
        s.set_min_level(int(levels[k]))
        assert np.array_equal(got[k], s.render(cams[k:k + 1], 40, 28)[0])
    s.set_min_level(0)
    # the rule, against its closed form: distance = |z_st - eye.z|
    z_st = wl.geometry(cfg)["z_st"]
    cam = np.array(cams[0], dtype=np.float32).reshape(16).copy()
    for d, want in ((0.5, 0), (1.0, 0), (1.99, 0), (2.0, 1), (3.9, 1), (4.0, 2), (8.0, 3), (1000.0, cfg.height)):
        cam[2] = z_st - d
        assert s.lod_levels(cam[None], 1.0)[0] == min(want, cfg.height), d
    assert s.lod_levels(cam[None], 0.0)[0] == 0
