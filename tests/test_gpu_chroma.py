"""GPU parity on chroma-subsampled streams (R18): the CUDA path through the C ABI against the oracle.

The streams come from the oracle's encoder (hmlfc_encode does not subsample); decoded pixels bit-exact, views within 1 LSB.
On these streams every entry point runs the chroma instantiation of its fast kernel (hmlfc_render, hmlfc_decode_views / _blocks: 4 x 4 blocks),
cross-checked against the per-sample kernels."""
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


def _subsampled_stream(name, tau):
    cfg = wl.CONFIGS[name]
    lf = wl.light_field(cfg)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, tau // 2, tau, geometry=wl.geometry(cfg),
                        seed=cfg.seed, chroma=1)
    tree = orc.Tree(lf, p)
    data = tree.serialize()
    tree.close()
    return cfg, lf, data, orc.Stream(data)


@pytest.mark.parametrize("name", CASES)
@pytest.mark.parametrize("tau", [0, 40])
def test_subsampled_stream_decode_and_render(P, name, tau):
    cfg = wl.CONFIGS[name]
    if (cfg.Ws // 2) % cfg.block or (cfg.Ht // 2) % cfg.block:
        pytest.skip("the block size does not tile the half-resolution planes")
    cfg, lf, data, s = _subsampled_stream(name, tau)
    h = P.hmlfc_load(data)
    coords = wl.all_coords(cfg)
    expect = s.decode(coords)
    for variant in (P.DECODE_AUTO, P.DECODE_THREAD, P.DECODE_QUEUE, P.DECODE_QUEUE_LAZY, P.DECODE_QUEUE_BLOCKREC):   # thread per coordinate, or the queue kernel's chroma instantiation
        P.hmlfc_set_decode_variant(h, variant)
        assert np.array_equal(P.hmlfc_decode(h, _dev(coords)).cpu().numpy(), expect), variant
    P.hmlfc_set_decode_variant(h, P.DECODE_AUTO)
    # whole views and whole blocks
    views = np.array([(u, v) for v in range(cfg.V) for u in range(cfg.U)], dtype=np.int32)
    got = P.hmlfc_decode_views(h, _dev(views)).cpu().numpy()
    assert np.array_equal(got.reshape(-1, 3), expect)
    rng = np.random.Generator(np.random.PCG64(cfg.seed + 77))
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
    # views
    cams = wl.camera_path(cfg)
    ref = s.render(cams, cfg.out_w, cfg.out_h)
    P.hmlfc_set_render_variant(h, P.RENDER_PIXEL)
    unshared = P.hmlfc_render(h, _dev(cams), cfg.out_w, cfg.out_h).cpu().numpy()
    # 4 x 4 blocks: the tile kernel's chroma instantiation (whatever fused variant is asked for); otherwise the thread-per-pixel kernel
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
    # the counting aid does not read these streams and says so
    with pytest.raises(P.HmlfcError):
        P.hmlfc_footprint_decode(h, _dev(coords[:16]))
    P.hmlfc_free(h)


def test_lossless_luma_and_subsampled_chroma(P):
    # tau = 0 on a subsampled stream: the decoded light field equals the numpy closed form of tests/test_oracle_chroma.py
    cfg, lf, data, s = _subsampled_stream("cfg1_lossy", 0)
    h = P.hmlfc_load(data)
    got = P.hmlfc_decode(h, _dev(wl.all_coords(cfg))).cpu().numpy().reshape(lf.shape)
    r, g, b = (lf[..., i].astype(np.int64) for i in range(3))
    co = r - b
    t = b + np.floor_divide(co, 2)
    cg = g - t
    y = t + np.floor_divide(cg, 2)

    def downup(p):
        q = p[..., 0::2, 0::2] + p[..., 0::2, 1::2] + p[..., 1::2, 0::2] + p[..., 1::2, 1::2]
        q = np.sign(q) * ((2 * np.abs(q) + 4) // 8)
        return np.repeat(np.repeat(q, 2, axis=-2), 2, axis=-1)

    co, cg = downup(co), downup(cg)
    t = y - np.floor_divide(cg, 2)
    g2 = cg + t
    b2 = t - np.floor_divide(co, 2)
    r2 = b2 + co
    assert np.array_equal(got, np.clip(np.stack([r2, g2, b2], axis=-1), 0, 255).astype(np.uint8))
    P.hmlfc_free(h)
