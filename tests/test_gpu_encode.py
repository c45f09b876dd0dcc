"""GPU parity of hmlfc_encode (the whole HMLFC encoder in CUDA kernels: colour + hierarchy, phase-shifted search, replacement step,
two block thresholds, BISE packing, BFS stream order -- PAPER.md:200-276) against the oracle's encoder: the two compressed streams
must be equal BYTE FOR BYTE (header, top-level RKVs, directory, flag maps, payload strings, motion-vector strings).  The two
writers share no code; the format is DESIGN.md section 4.  Streams fed to the decode / render tests still come from the oracle only."""
import struct

import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def P():
    import paper_1902_09396_b200 as pkg

    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    return pkg


def _section(data, off):
    names = ("rkv", "directory", "flags", "payload", "mv", "end")
    offs = struct.unpack_from("<6Q", data, 112)
    where = "header"
    for n, o in zip(names, offs):
        if off >= o:
            where = n
    return where


def _assert_same_stream(got, expect):
    if got == expect:
        return
    a, b = np.frombuffer(got, np.uint8), np.frombuffer(expect, np.uint8)
    n = min(len(a), len(b))
    diff = np.nonzero(a[:n] != b[:n])[0]
    first = int(diff[0]) if len(diff) else n
    raise AssertionError(f"streams differ: lengths {len(a)} / {len(b)}, {len(diff)} bytes differ, first at {first} "
                         f"(section {_section(expect, first)}), header offsets {struct.unpack_from('<6Q', expect, 112)}")


def _gpu_encode(P, cfg, lf, tau_ref, tau_res, policy=0):
    return P.hmlfc_encode(torch.from_numpy(lf).cuda(), cfg.height, cfg.block, cfg.window, tau_ref, tau_res, policy,
                          geometry=wl.geometry(cfg), seed=cfg.seed)


@pytest.mark.parametrize("name", ["cfg1", "cfg1_lossy", "mini2", "mini3", "mini4", "mini_b2", "mini_b8", "mini_h8", "mini_w64"])
def test_encoded_stream_equals_the_oracle_stream(P, enc, name):
    # cfg1: tau = 0 (every block kept); mini3: odd 5 x 5 grid (partial clusters); mini_b2 / mini_b8: B = 2 / 8, W = 5 / 8; mini_h8 / mini_w64:
    # the format's limits, tree height 8 and search window 64
    cfg, lf, data, info, s = enc(name)
    got, stats = _gpu_encode(P, cfg, lf, info["tau_ref"], info["tau_res"])
    _assert_same_stream(got, data)
    assert stats["n_plane_channels"] == struct.unpack_from("<Q", data, 104)[0]
    assert stats["kernel_launches"] >= cfg.height + 5
    # the encoder's own reconstruction error (a kernel over its planes) = the oracle's P1 reconstruction error, exactly
    sse = int(((info["p1"].astype(np.int64) - lf.astype(np.int64)) ** 2).sum())
    assert stats["sse"] == sse and (stats["tau_ref"], stats["tau_res"]) == (info["tau_ref"], info["tau_res"])
    assert stats["psnr"] == info["psnr"] or abs(stats["psnr"] - info["psnr"]) < 1e-9


@pytest.mark.parametrize("policy", [orc.POLICY_ALL, orc.POLICY_LITERAL, orc.POLICY_NOMOTION])
@pytest.mark.parametrize("tau", [0, 37, 100000])
def test_other_policies_and_degenerate_thresholds(P, policy, tau):
    # tau = 100000: no block survives (empty payload and, under `literal`, empty motion-vector strings)
    cfg = wl.CONFIGS["mini3"]
    lf = wl.light_field(cfg)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, tau // 2, tau, policy=policy,
                        geometry=wl.geometry(cfg), seed=cfg.seed)
    data, info, tree = orc.encode(lf, p)
    tree.close()
    got, _ = _gpu_encode(P, cfg, lf, tau // 2, tau, policy)
    _assert_same_stream(got, data)


def test_encoded_stream_loads_and_decodes_to_the_oracle_reconstruction(P, enc):
    cfg, lf, data, info, s = enc("mini4")
    got, _ = _gpu_encode(P, cfg, lf, info["tau_ref"], info["tau_res"])
    h = P.hmlfc_load(got)
    coords = wl.all_coords(cfg)
    out = P.hmlfc_decode(h, torch.from_numpy(coords).cuda()).cpu().numpy()
    assert np.array_equal(out.reshape(info["p1"].shape), info["p1"])  # = the oracle encoder's own reconstruction (P1)
    P.hmlfc_free(h)


def _full_configs():
    import os

    extra = [c for c in os.environ.get("HMLFC_FULL", "").split(",") if c]
    return ["cfg2", "cfg3"] + [c for c in ("cfg4", "cfg5") if c in extra]


@pytest.mark.parametrize("name", _full_configs())
def test_full_size_stream_equals_the_oracle_stream(P, name):
    """BASELINE.json configs[1..4] at full size: the GPU encoder's stream against the oracle encoder's cached stream (cfg2: 7.5 MB,
    cfg3: 82 MB, cfg4: 175 MB, cfg5: 1.04 GB).  cfg2 and cfg3 always run; cfg4 / cfg5 when HMLFC_FULL names them (the oracle needs
    ~75 s / ~8 min on 16 cores for what the GPU encoder does in 0.26 s / 1.6 s; results recorded in profiles/r01_all_configs.md)."""
    from oracle import streams

    cfg, data, info = streams.get_stream(name)
    lf = wl.light_field(cfg)
    got, stats = _gpu_encode(P, cfg, lf, info["tau_ref"], info["tau_res"])
    del lf
    P.hmlfc_encode_release_scratch()
    _assert_same_stream(got, data)
    n_pairs = sum((((cfg.U - 1) >> L) + 1) * (((cfg.V - 1) >> L) + 1) - ((((cfg.U - 1) >> L) + 2) // 2) * ((((cfg.V - 1) >> L) + 2) // 2)
                  for L in range(cfg.height))
    assert stats["n_search_blocks"] == 3 * n_pairs * (cfg.Ws // cfg.block) * (cfg.Ht // cfg.block)


@pytest.mark.parametrize("name,target", [("mini2", 38.0), ("mini3", 43.5), ("mini_b8", 36.0), ("cfg1", 120.0)])
def test_threshold_bisection_to_a_psnr_target_reproduces_the_oracle(P, name, target):
    # PAPER.md:375; the oracle's encode(lf, p, target) bisects tau_res on its P1 reconstruction; hmlfc_encode_psnr must take the same
    # decisions (same PSNR values, same steps) and write the same stream.  cfg1 at 120 dB: unreachable, ends at the smallest tau
    cfg = wl.CONFIGS[name]
    lf = wl.light_field(cfg)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, 0, 0, geometry=wl.geometry(cfg), seed=cfg.seed)
    data, info, tree = orc.encode(lf, p, target)
    tree.close()
    got, stats = P.hmlfc_encode(torch.from_numpy(lf).cuda(), cfg.height, cfg.block, cfg.window, geometry=wl.geometry(cfg), seed=cfg.seed,
                                target_psnr=target)
    assert (stats["tau_ref"], stats["tau_res"]) == (info["tau_ref"], info["tau_res"])
    assert stats["psnr"] == info["psnr"] or abs(stats["psnr"] - info["psnr"]) < 1e-9
    assert 1 <= stats["bisection_steps"] <= 12
    _assert_same_stream(got, data)


def test_cfg2_bisection_to_40_db_reproduces_the_cached_oracle_stream(P):
    from oracle import streams

    cfg, data, info = streams.get_stream("cfg2")
    got, stats = P.hmlfc_encode(torch.from_numpy(wl.light_field(cfg)).cuda(), cfg.height, cfg.block, cfg.window, geometry=wl.geometry(cfg),
                                seed=cfg.seed, target_psnr=cfg.target_psnr)
    assert stats["tau_res"] == info["tau_res"] and abs(stats["psnr"] - info["psnr"]) < 1e-9
    _assert_same_stream(got, data)


def test_invalid_and_unsupported_arguments(P):
    lf = torch.zeros((2, 2, 16, 16, 3), dtype=torch.uint8, device="cuda")
    with pytest.raises(P.HmlfcError):
        P.hmlfc_encode(lf, 1, block=3)          # B must be 2, 4 or 8
    with pytest.raises(P.HmlfcError):
        P.hmlfc_encode(lf, 9)                   # height > 8
    with pytest.raises(P.HmlfcError):
        P.hmlfc_encode(lf, 1, tau_res=-1)
    with pytest.raises(P.HmlfcError):
        P.hmlfc_encode(lf, 1, target_psnr=-3.0)
    with pytest.raises(P.HmlfcError):
        P.hmlfc_encode(lf, 1, target_psnr=40.0, max_iter=0)


@pytest.mark.parametrize("U,V,Ws,Ht,h,B,W", [(1, 1, 8, 4, 1, 4, 16), (2, 1, 8, 8, 1, 4, 3), (1, 3, 12, 8, 2, 2, 2), (3, 3, 16, 8, 3, 8, 1), (2, 2, 4, 4, 1, 4, 0)])
def test_degenerate_shapes(P, U, V, Ws, Ht, h, B, W):
    """One view (no predictive plane at all), one row / column of views, one block per image, a window far wider than the image, W = 0
    (prediction from the co-located block only): encoder stream equal to the oracle's, and the decode of every pixel through the GPU-
    encoded stream equal to the oracle's decode."""
    from conftest import random_lf

    lf = random_lf(np.random.default_rng(U * 100 + V * 10 + B), U, V, Ws, Ht)
    for tau in (0, 25):
        p = orc.make_params(U, V, Ws, Ht, h, B, W, tau // 2, tau, seed=7)
        data, info, tree = orc.encode(lf, p)
        tree.close()
        got, stats = P.hmlfc_encode(torch.from_numpy(lf).cuda(), h, B, W, tau // 2, tau, seed=7)
        _assert_same_stream(got, data)
        hd = P.hmlfc_load(got)
        views = np.array([[u, v] for v in range(V) for u in range(U)], dtype=np.int32)
        dec = P.hmlfc_decode_views(hd, torch.from_numpy(views).cuda()).cpu().numpy().reshape(V, U, Ht, Ws, 3)
        assert np.array_equal(dec, orc.Stream(data).decode_full())
        if tau == 0:
            assert np.array_equal(dec, lf)  # lossless round trip (north_star pin 1)
        # a camera ON the camera plane (so that a 1-view-wide grid is hit at all), looking at the centre of the image plane
        ex, ey = 0.4 * (U - 1), 0.3 * (V - 1)
        cam = np.zeros((1, 16), dtype=np.float32)
        cam[0, 0:3] = (ex, ey, 0.0)
        cam[0, 3:6], cam[0, 6:9] = (1, 0, 0), (0, 1, 0)
        cam[0, 9:12] = ((Ws - 1) / 2 - ex, (Ht - 1) / 2 - ey, 1.0)
        cam[0, 12:14] = (0.45 * Ws, 0.45 * Ht)
        ref = orc.Stream(data).render(cam, 40, 24)
        assert ref.any()
        outs = []
        for variant in (P.RENDER_AUTO, P.RENDER_PIXEL, P.RENDER_WARP, *P.RENDER_FUSED):
            P.hmlfc_set_render_variant(hd, variant)
            outs.append(P.hmlfc_render(hd, torch.from_numpy(cam).cuda(), 40, 24).cpu().numpy())
            assert np.abs(outs[-1].astype(int) - ref.astype(int)).max() <= 1, variant
            assert np.array_equal(outs[-1], outs[0])
        P.hmlfc_free(hd)


def test_more_than_65535_plane_channels(P):
    """160 x 160 views of 4 x 4 pixels, h = 2: 96,000 plane-channels, more than one grid.y's worth -- the encoder's kernels run in
    chunks of 65,535 plane-channels.  Stream equal to the oracle's; every view decodes to the oracle's decode."""
    U = V = 160
    rng = np.random.default_rng(11)
    base = rng.integers(0, 256, (V + 4, U + 4, 3)).astype(np.float64)
    lf = np.empty((V, U, 4, 4, 3), dtype=np.uint8)
    for t in range(4):
        for s in range(4):  # neighbouring views are shifted copies of one image: inter-view coherence
            lf[:, :, t, s] = np.clip(base[t:t + V, s:s + U] + rng.normal(0, 3.0, (V, U, 3)), 0, 255).astype(np.uint8)
    geo = dict(uv_origin=(0.0, 0.0), uv_step=(0.02, 0.02), st_origin=(0.0, 0.0), st_step=(1.0, 1.0), z_st=1.0)  # a dense camera grid
    p = orc.make_params(U, V, 4, 4, 2, 4, 1, 6, 12, geometry=geo, seed=3)
    data, info, tree = orc.encode(lf, p)
    tree.close()
    assert struct.unpack_from("<Q", data, 104)[0] == 96000
    got, stats = P.hmlfc_encode(torch.from_numpy(lf).cuda(), 2, 4, 1, 6, 12, geometry=geo, seed=3)
    _assert_same_stream(got, data)
    h = P.hmlfc_load(got)
    views = np.array([[u, v] for v in range(V) for u in range(U)], dtype=np.int32)
    dec = P.hmlfc_decode_views(h, torch.from_numpy(views).cuda()).cpu().numpy().reshape(V, U, 4, 4, 3)
    assert np.array_equal(dec, orc.Stream(data).decode_full())
    # a camera behind the camera plane: every 32 x 32 output tile spans dozens of views (more than the CTA kernel's 4 x 4 per pass),
    # so the tile is split down to direct decodes; all render kernels agree with the oracle and with one another
    cam = np.zeros((1, 16), dtype=np.float32)
    cam[0, 0:3] = (1.6, 1.55, -40.0)
    cam[0, 3:6], cam[0, 6:9] = (1, 0, 0), (0, 1, 0)
    cam[0, 9:12] = ((1.5 - 1.6) / 41.0, (1.5 - 1.55) / 41.0, 1.0)
    cam[0, 12:14] = (1.4 / 41.0, 1.4 / 41.0)
    s_or = orc.Stream(data)
    ref = s_or.render(cam, 96, 64)
    assert ref.any()
    first = None
    for variant in (P.RENDER_AUTO, P.RENDER_PIXEL, P.RENDER_WARP, *P.RENDER_FUSED):
        P.hmlfc_set_render_variant(h, variant)
        out = P.hmlfc_render(h, torch.from_numpy(cam).cuda(), 96, 64).cpu().numpy()
        assert np.abs(out.astype(int) - ref.astype(int)).max() <= 1, variant
        first = out if first is None else first
        assert np.array_equal(out, first)
    P.hmlfc_free(h)


def test_randomised_shapes_and_parameters(P):
    """150 seeded random small light fields (grid 1..6 x 1..6, images of 1..6 x 1..5 blocks, B in {2,4,8}, h 1..4, W 0..9, thresholds 0..120,
    all three policies): GPU encoder stream = oracle stream; GPU decode of every view (dense kernels) and of shuffled coordinates (both
    decode kernels) = oracle decode; one on-plane view through every render kernel within 1 LSB of the oracle and byte-identical."""
    from conftest import random_lf

    rng = np.random.default_rng(20260411)
    for case in range(150):
        B = int(rng.choice([2, 4, 8]))
        U, V = int(rng.integers(1, 7)), int(rng.integers(1, 7))
        Ws, Ht = B * int(rng.integers(1, 7)), B * int(rng.integers(1, 6))
        if Ws % 4:
            Ws *= 2  # hmlfc_hierarchy needs Ws % 4 == 0
        h, W, tau, policy = int(rng.integers(1, 5)), int(rng.integers(0, 10)), int(rng.integers(0, 121)), int(rng.integers(0, 4))
        tag = (case, U, V, Ws, Ht, h, B, W, tau, policy)
        lf = random_lf(rng, U, V, Ws, Ht, smooth=bool(case & 1))
        p = orc.make_params(U, V, Ws, Ht, h, B, W, tau // 2, tau, policy=policy, seed=case)
        data, info, tree = orc.encode(lf, p)
        tree.close()
        got, stats = P.hmlfc_encode(torch.from_numpy(lf).cuda(), h, B, W, tau // 2, tau, policy, seed=case)
        assert got == data, tag
        s = orc.Stream(data)
        full = s.decode_full()
        hd = P.hmlfc_load(got)
        views = np.array([[u, v] for v in range(V) for u in range(U)], dtype=np.int32)
        for variant in (P.DECODE_AUTO, P.DECODE_QUEUE, P.DECODE_QUEUE_LAZY, P.DECODE_QUEUE_BLOCKREC):
            P.hmlfc_set_decode_variant(hd, variant)
            dec = P.hmlfc_decode_views(hd, torch.from_numpy(views).cuda()).cpu().numpy().reshape(V, U, Ht, Ws, 3)
            assert np.array_equal(dec, full), tag
        coords = np.stack([a.ravel() for a in np.meshgrid(np.arange(U), np.arange(V), np.arange(Ws), np.arange(Ht), indexing="ij")], 1).astype(np.int32)
        coords = coords[rng.permutation(len(coords))]
        expect = full[coords[:, 1], coords[:, 0], coords[:, 3], coords[:, 2]]
        for variant in (P.DECODE_THREAD, P.DECODE_QUEUE, P.DECODE_QUEUE_LAZY, P.DECODE_QUEUE_BLOCKREC):
            P.hmlfc_set_decode_variant(hd, variant)
            assert np.array_equal(P.hmlfc_decode(hd, torch.from_numpy(coords).cuda()).cpu().numpy(), expect), tag
        blocks = np.stack([a.ravel() for a in np.meshgrid(np.arange(U), np.arange(V), np.arange(Ws // B), np.arange(Ht // B), indexing="ij")], 1).astype(np.int32)
        blocks = blocks[rng.permutation(len(blocks))]
        bexp = np.stack([full[b[1], b[0], b[3] * B:(b[3] + 1) * B, b[2] * B:(b[2] + 1) * B] for b in blocks])
        for variant in (P.DECODE_AUTO, P.DECODE_QUEUE, P.DECODE_QUEUE_LAZY, P.DECODE_QUEUE_BLOCKREC):
            P.hmlfc_set_decode_variant(hd, variant)
            assert np.array_equal(P.hmlfc_decode_blocks(hd, torch.from_numpy(blocks).cuda()).cpu().numpy(), bexp), tag
        P.hmlfc_set_decode_variant(hd, P.DECODE_AUTO)
        cam = np.zeros((1, 16), dtype=np.float32)
        ex, ey = float(rng.uniform(0, max(U - 1, 0))), float(rng.uniform(0, max(V - 1, 0)))
        cam[0, 0:3] = (ex, ey, 0.0)
        cam[0, 3:6], cam[0, 6:9] = (1, 0, 0), (0, 1, 0)
        cam[0, 9:12] = ((Ws - 1) / 2 - ex, (Ht - 1) / 2 - ey, 1.0)
        cam[0, 12:14] = (0.55 * Ws, 0.55 * Ht)   # a little wider than the image plane: the border rays miss
        ref = s.render(cam, 45, 37)
        first = None
        for variant in (P.RENDER_AUTO, P.RENDER_PIXEL, P.RENDER_WARP, P.RENDER_WARP8, *P.RENDER_FUSED):
            P.hmlfc_set_render_variant(hd, variant)
            out = P.hmlfc_render(hd, torch.from_numpy(cam).cuda(), 45, 37).cpu().numpy()
            assert np.abs(out.astype(int) - ref.astype(int)).max() <= 1, (tag, variant)
            first = out if first is None else first
            assert np.array_equal(out, first), (tag, variant)
        P.hmlfc_free(hd)
