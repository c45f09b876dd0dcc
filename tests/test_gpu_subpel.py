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
