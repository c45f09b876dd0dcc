"""GPU parity on streams with half-pel motion compensation (R28): the CUDA path through the C ABI against the oracle.

The streams come from the oracle's encoder (hmlfc_encode searches whole pixels); decoded pixels bit-exact, views within 1 LSB.
On these streams hmlfc_decode / _views / _blocks and hmlfc_render run the per-sample kernels."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

CASES = ["cfg1_lossy", "mini2", "mini3", "mini_b2", "mini_b8", "mini_h8"]


@pytest.fixture(scope="module")
def P():
    import paper_1902_09396_b200 as pkg

    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    return pkg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _halfpel_stream(name, tau, chroma=0):
    cfg = wl.CONFIGS[name]
    lf = wl.light_field(cfg)
    # (window 4: the oracle's half-pel search is exhaustive over (4W + 1)^2 interpolated candidates)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, min(cfg.window, 4), tau // 2, tau, geometry=wl.geometry(cfg),
                        seed=cfg.seed, chroma=chroma, subpel=1)
    tree = orc.Tree(lf, p)
    data = tree.serialize()
    tree.close()
    return cfg, lf, data, orc.Stream(data)


@pytest.mark.parametrize("name", CASES)
@pytest.mark.parametrize("tau", [0, 40])
def test_halfpel_stream_decode_and_render(P, name, tau):
    cfg, lf, data, s = _halfpel_stream(name, tau)
    assert data[55] == 1
    h = P.hmlfc_load(data)
    coords = wl.all_coords(cfg)
    expect = s.decode(coords)
    if tau == 0:
        assert np.array_equal(expect.reshape(lf.shape), lf)
    for variant in (P.DECODE_AUTO, P.DECODE_THREAD, P.DECODE_QUEUE, P.DECODE_QUEUE_LAZY, P.DECODE_QUEUE_BLOCKREC):   # thread per coordinate, or the queue kernel's half-pel instantiation
        P.hmlfc_set_decode_variant(h, variant)
        assert np.array_equal(P.hmlfc_decode(h, _dev(coords)).cpu().numpy(), expect), variant
    P.hmlfc_set_decode_variant(h, P.DECODE_AUTO)
    views = np.array([(u, v) for v in range(cfg.V) for u in range(cfg.U)], dtype=np.int32)
    assert np.array_equal(P.hmlfc_decode_views(h, _dev(views)).cpu().numpy().reshape(-1, 3), expect)
    rng = np.random.Generator(np.random.PCG64(cfg.seed + 78))
    nb = 200
    blocks = np.stack([rng.integers(0, cfg.U, nb), rng.integers(0, cfg.V, nb), rng.integers(0, cfg.Ws // cfg.block, nb),
                       rng.integers(0, cfg.Ht // cfg.block, nb)], axis=1).astype(np.int32)
    B = cfg.block
    bc = np.array([(u, v, bx * B + i, by * B + j) for (u, v, bx, by) in blocks for j in range(B) for i in range(B)], dtype=np.int32)
    assert np.array_equal(P.hmlfc_decode_blocks(h, _dev(blocks)).cpu().numpy().reshape(-1, 3), s.decode(bc))
    P.hmlfc_set_decode_variant(h, P.DECODE_THREAD)   # whole views and blocks once more through the per-sample kernel (4 x 4 blocks: above ran the block-row kernel)
    assert np.array_equal(P.hmlfc_decode_views(h, _dev(views)).cpu().numpy().reshape(-1, 3), expect)
    assert np.array_equal(P.hmlfc_decode_blocks(h, _dev(blocks)).cpu().numpy().reshape(-1, 3), s.decode(bc))
    P.hmlfc_set_decode_variant(h, P.DECODE_AUTO)
    cams = wl.camera_path(cfg)
    ref = s.render(cams, cfg.out_w, cfg.out_h)
    P.hmlfc_set_render_variant(h, P.RENDER_PIXEL)
    unshared = P.hmlfc_render(h, _dev(cams), cfg.out_w, cfg.out_h).cpu().numpy()
    # 4 x 4 blocks: the tile kernel's half-pel instantiation (whatever fused variant is asked for); otherwise the thread-per-pixel kernel
    for variant in (P.RENDER_AUTO, P.RENDER_TILES, P.RENDER_TILES_W256X3, P.RENDER_CTA, P.RENDER_CTA_BIG, P.RENDER_WARP):
        P.hmlfc_set_render_variant(h, variant)
        out = P.hmlfc_render(h, _dev(cams), cfg.out_w, cfg.out_h).cpu().numpy()
        d = np.abs(out.astype(np.int16) - ref.astype(np.int16))
        assert d.max() <= 1 and (d > 0).mean() < 1e-3, (variant, int(d.max()))
        assert np.array_equal(out, unshared), variant
    # a magnified, rotated batch (several tiles per view, ragged edges) and every progressive level
    cams2 = wl.camera_path(cfg, n_views=3, out_w=200, out_h=136, seed_offset=3)
    for level in range(cfg.height + 1):
        P.hmlfc_set_min_level(h, level)
        P.hmlfc_set_render_variant(h, P.RENDER_PIXEL)
        a = P.hmlfc_render(h, _dev(cams2), 200, 136)
        P.hmlfc_set_render_variant(h, P.RENDER_AUTO)
        b = P.hmlfc_render(h, _dev(cams2), 200, 136)
        assert torch.equal(a, b), level
    P.hmlfc_set_min_level(h, 0)
    with pytest.raises(P.HmlfcError):   # the counting aid does not read these streams and says so
        P.hmlfc_footprint_decode(h, _dev(coords[:16]))
    P.hmlfc_free(h)


def test_halfpel_with_subsampled_chroma_and_progressive_levels(P):
    cfg, lf, data, s = _halfpel_stream("mini3", 30, chroma=1)
    h = P.hmlfc_load(data)
    coords = wl.random_coords(cfg, 20_001)
    views = np.array([(u, v) for v in range(cfg.V) for u in range(cfg.U)], dtype=np.int32)
    allc = wl.all_coords(cfg)
    for level in range(cfg.height + 1):
        s.set_min_level(level)
        P.hmlfc_set_min_level(h, level)
        assert np.array_equal(P.hmlfc_decode(h, _dev(coords)).cpu().numpy(), s.decode(coords)), level
        # whole views: the block-row kernel's instantiation for both flags at once
        assert np.array_equal(P.hmlfc_decode_views(h, _dev(views)).cpu().numpy().reshape(-1, 3), s.decode(allc)), level
    s.set_min_level(0)
    P.hmlfc_free(h)


def test_halfpel_offsets_at_the_image_border(P):
    # tau = 0 on a tiny light field with a window as large as the image: half-pel positions outside the image read zeros
    rng = np.random.Generator(np.random.PCG64(5))
    lf = rng.integers(0, 256, (2, 2, 8, 8, 3), dtype=np.uint8)
    p = orc.make_params(2, 2, 8, 8, 1, 4, 4, 0, 0, orc.POLICY_ALL, subpel=1)
    tree = orc.Tree(lf, p)
    data = tree.serialize()
    tree.close()
    s = orc.Stream(data)
    h = P.hmlfc_load(data)
    coords = np.array([(u, v, x, y) for v in range(2) for u in range(2) for y in range(8) for x in range(8)], dtype=np.int32)
    got = P.hmlfc_decode(h, _dev(coords)).cpu().numpy()
    assert np.array_equal(got, s.decode(coords)) and np.array_equal(got.reshape(lf.shape), lf)
    P.hmlfc_free(h)


def test_randomised_chroma_and_halfpel_streams(P):
    """48 seeded random cases: small light fields (2..6 x 2..6 views of 16..48-pixel images, B in {2, 4, 8}, h 1..3, W 1..4, thresholds
    0..60, three policies) with the chroma flag, the half-pel flag or both, a random slab geometry, a random progressive level and two
    rotated cameras: every decode entry point bit-exact against the oracle (fast and per-sample kernels), every render variant within
    1 LSB of the oracle and byte-identical to the thread-per-pixel kernel."""
    from conftest import random_lf

    rng = np.random.default_rng(19020939)
    n_fast = 0
    for case in range(48):
        B = int(rng.choice([4, 4, 4, 2, 8]))
        chroma, subpel = [(1, 0), (0, 1), (1, 1)][case % 3]
        U, V = int(rng.integers(2, 7)), int(rng.integers(2, 7))
        unit = 2 * B if chroma else B
        Ws, Ht = unit * int(rng.integers(max(1, 16 // unit), 48 // unit + 1)), unit * int(rng.integers(max(1, 16 // unit), 48 // unit + 1))
        h, W, tau = int(rng.integers(1, 4)), int(rng.integers(1, 5)), int(rng.integers(0, 60))
        policy = int(rng.choice([orc.POLICY_ADAPTIVE, orc.POLICY_ALL, orc.POLICY_LITERAL]))
        step_u, step_v = float(rng.uniform(0.2, 1.0)) * Ws / (2 * U), float(rng.uniform(0.2, 1.0)) * Ht / (2 * V)
        z_st = float(rng.uniform(0.3, 2.0)) * Ws
        geo = dict(uv_origin=(float(rng.uniform(-3, 3)), float(rng.uniform(-3, 3))), uv_step=(step_u, step_v),
                   st_origin=(float(rng.uniform(-5, 5)), float(rng.uniform(-5, 5))), st_step=(float(rng.uniform(0.5, 2.0)), float(rng.uniform(0.5, 2.0))),
                   z_st=z_st)
        lf = random_lf(rng, U, V, Ws, Ht)
        p = orc.make_params(U, V, Ws, Ht, h, B, W, tau // 2, tau, policy, geometry=geo, seed=case, chroma=chroma, subpel=subpel)
        tree = orc.Tree(lf, p)
        data = tree.serialize()
        tree.close()
        s = orc.Stream(data)
        hd = P.hmlfc_load(data)
        L = int(rng.integers(0, h + 1))
        s.set_min_level(L)
        P.hmlfc_set_min_level(hd, L)
        tag = (case, B, chroma, subpel, h, W, tau, policy, L)
        # decode: every coordinate, whole views, random blocks -- default (fast) kernels and the per-sample ones
        coords = np.array([(u, v, x, y) for v in range(V) for u in range(U) for y in range(Ht) for x in range(Ws)], dtype=np.int32)
        expect = s.decode(coords)
        views = np.array([(u, v) for v in range(V) for u in range(U)], dtype=np.int32)
        nb = 64
        blocks = np.stack([rng.integers(0, U, nb), rng.integers(0, V, nb), rng.integers(0, Ws // B, nb), rng.integers(0, Ht // B, nb)], axis=1).astype(np.int32)
        bc = np.array([(u, v, bx * B + i, by * B + j) for (u, v, bx, by) in blocks for j in range(B) for i in range(B)], dtype=np.int32)
        bexp = s.decode(bc)
        for variant in (P.DECODE_AUTO, P.DECODE_THREAD):
            P.hmlfc_set_decode_variant(hd, variant)
            assert np.array_equal(P.hmlfc_decode(hd, _dev(coords)).cpu().numpy(), expect), tag + (variant, "decode")
            assert np.array_equal(P.hmlfc_decode_views(hd, _dev(views)).cpu().numpy().reshape(-1, 3), expect), tag + (variant, "views")
            assert np.array_equal(P.hmlfc_decode_blocks(hd, _dev(blocks)).cpu().numpy().reshape(-1, 3), bexp), tag + (variant, "blocks")
        P.hmlfc_set_decode_variant(hd, P.DECODE_AUTO)
        # render: two rotated off-plane cameras
        uc = (geo["uv_origin"][0] + 0.5 * (U - 1) * step_u, geo["uv_origin"][1] + 0.5 * (V - 1) * step_v)
        sc = (geo["st_origin"][0] + 0.5 * (Ws - 1) * geo["st_step"][0], geo["st_origin"][1] + 0.5 * (Ht - 1) * geo["st_step"][1])
        cams = []
        for _ in range(2):
            eye = (uc[0] + rng.uniform(-0.35, 0.35) * U * step_u, uc[1] + rng.uniform(-0.35, 0.35) * V * step_v, -float(rng.uniform(0.0, 0.8)) * z_st)
            look = (sc[0] + rng.uniform(-0.3, 0.3) * Ws * geo["st_step"][0], sc[1] + rng.uniform(-0.3, 0.3) * Ht * geo["st_step"][1], z_st)
            d = float(np.linalg.norm(np.array(look) - np.array(eye)))
            th = float(rng.uniform(0.1, 0.5)) * Ws * geo["st_step"][0] / d
            cams.append(wl._camera(eye, look, th, th * float(rng.uniform(0.6, 1.4))))
        cams = np.stack(cams)
        Wo, Ho = int(rng.integers(20, 100)), int(rng.integers(20, 80))
        ref = s.render(cams, Wo, Ho)
        P.hmlfc_set_render_variant(hd, P.RENDER_PIXEL)
        unshared = P.hmlfc_render(hd, _dev(cams), Wo, Ho).cpu().numpy()
        assert np.abs(unshared.astype(int) - ref.astype(int)).max() <= 1, tag
        for variant in (P.RENDER_AUTO, P.RENDER_TILES, P.RENDER_CTA_SMALL, P.RENDER_WARP):
            P.hmlfc_set_render_variant(hd, variant)
            assert np.array_equal(P.hmlfc_render(hd, _dev(cams), Wo, Ho).cpu().numpy(), unshared), tag + (variant,)
        n_fast += int(B == 4)
        P.hmlfc_free(hd)
    assert n_fast >= 20   # most cases ran the instantiations of the fast kernels (4 x 4 blocks)
