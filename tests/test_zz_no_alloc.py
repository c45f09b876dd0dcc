"""hmlfc_render_noalloc (include/hmlfc.h): the render entry point that allocates nothing -- tile tables in the library's static device
buffer instead of scratch memory from a pool -- against the existing hmlfc_render, byte for byte (the bar every render variant meets in
tests/test_gpu_parity.py), on calls in a row that share the buffer.

Collected last on purpose (the file name): a failure here must not hide other tests under `pytest -x`."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def P():
    import paper_1902_09396_b200 as pkg

    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    return pkg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _existing(P, h, cams, W, H):
    """The existing paths: the default choice of hmlfc_render, the tile kernel with pool scratch, and the unshared definition."""
    outs = []
    for variant in (P.RENDER_AUTO, P.RENDER_TILES, P.RENDER_PIXEL):
        P.hmlfc_set_render_variant(h, variant)
        outs.append(P.hmlfc_render(h, cams, W, H).clone())
    P.hmlfc_set_render_variant(h, P.RENDER_AUTO)
    assert torch.equal(outs[0], outs[1]) and torch.equal(outs[0], outs[2])
    return outs[0]


def test_render_noalloc_equals_render_on_calls_in_a_row(P, enc):
    cfg, lf, data, info, s = enc("mini2")
    h = P.hmlfc_load(data)
    # three batches of different shapes through the one buffer, the large one first so that the later calls find its tables in it:
    # 12 views of 256 x 192 (32 x 32 tiles: 576 of them), 3 views of 200 x 136 (ragged edges), 2 views of 1024 x 832 on the camera
    # plane (>= 8x magnification: 64 x 32 tiles)
    batches = [(wl.camera_path(cfg, n_views=12, out_w=256, out_h=192), 256, 192),
               (wl.camera_path(cfg, n_views=3, seed_offset=5), cfg.out_w, cfg.out_h),
               (wl.camera_path(cfg, n_views=2, out_w=1024, out_h=832, on_plane=True), 1024, 832)]
    cams = [_dev(c) for c, _, _ in batches]
    refs = [_existing(P, h, c, W, H) for c, (_, W, H) in zip(cams, batches)]
    outs = [torch.full_like(r, 0xAB) for r in refs]
    # the calls, back to back on one stream, twice over (the second round starts from the first round's leftovers)
    for rnd in range(2):
        for o in outs:
            o.fill_(0xAB)
        for c, o, (_, W, H) in zip(cams, outs, batches):
            P.hmlfc_render_noalloc(h, c, W, H, out=o)
        torch.cuda.synchronize()
        for k, (o, r) in enumerate(zip(outs, refs)):
            assert torch.equal(o, r), (rnd, k, int((o != r).sum().item()))
    # and against the oracle, at the tolerance of the render parity tests (<= 1 LSB)
    ref = s.render(batches[1][0], cfg.out_w, cfg.out_h)
    d = np.abs(outs[1].cpu().numpy().astype(np.int16) - ref.astype(np.int16))
    assert d.max() <= 1 and (d > 0).mean() < 1e-3
    # no device memory is taken by the calls (kernels loaded and buffers made above): free memory does not fall across them
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for c, o, (_, W, H) in zip(cams, outs, batches):
        P.hmlfc_render_noalloc(h, c, W, H, out=o)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)
    P.hmlfc_free(h)


def test_render_noalloc_limit_and_arguments(P, enc):
    cfg, lf, data, info, s = enc("mini2")
    h = P.hmlfc_load(data)
    W = H = 512
    tile_w = 64 if W * H >= 8 * cfg.Ws * cfg.Ht else 32   # the documented rule (include/hmlfc.h)
    per_view = -(-W // tile_w) * -(-H // 32)
    n_fit = P.NOALLOC_MAX_TILES // per_view               # this many views fill the buffer
    assert n_fit * per_view == P.NOALLOC_MAX_TILES
    cams = _dev(wl.camera_path(cfg, n_views=n_fit + 1, out_w=W, out_h=H))
    out = torch.full((n_fit + 1, H, W, 3), 0xCD, dtype=torch.uint8, device="cuda")
    with pytest.raises(P.HmlfcError) as e:
        P.hmlfc_render_noalloc(h, cams, W, H, out=out)  # one view too many: a clear error, nothing launched
    assert e.value.code == -9
    torch.cuda.synchronize()
    assert bool((out == 0xCD).all())
    # exactly at the limit it renders, and equals hmlfc_render
    P.hmlfc_render_noalloc(h, cams[:n_fit], W, H, out=out[:n_fit])
    assert torch.equal(out[:n_fit], P.hmlfc_render(h, cams[:n_fit], W, H))
    # an empty batch is a no-op
    P.hmlfc_render_noalloc(h, cams[:0], W, H, out=out[:0])
    P.hmlfc_free(h)


@pytest.mark.parametrize("kind", ["chroma", "halfpel"])
def test_render_noalloc_on_chroma_and_halfpel_streams(P, kind):
    import oracle as orc

    cfg = wl.CONFIGS["mini3"]
    lf = wl.light_field(cfg)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, min(cfg.window, 4), 15, 30, geometry=wl.geometry(cfg), seed=cfg.seed,
                        chroma=1 if kind == "chroma" else 0, subpel=1 if kind == "halfpel" else 0)
    tree = orc.Tree(lf, p)
    data = tree.serialize()
    tree.close()
    h = P.hmlfc_load(data)
    cams = _dev(wl.camera_path(cfg, n_views=4, out_w=320, out_h=200))   # > 8x the light-field image: still 32 x 32 tiles on these streams
    ref = _existing(P, h, cams, 320, 200)
    out = torch.full_like(ref, 0xAB)
    for _ in range(2):
        out.fill_(0xAB)
        P.hmlfc_render_noalloc(h, cams, 320, 200, out=out)
        assert torch.equal(out, ref)
    P.hmlfc_free(h)
