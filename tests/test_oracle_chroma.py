"""Pins for the oracle's chroma subsampling ("the chroma channels are sub-sampled"; R18; SPEC.md:75-78:
2 x 2 box mean rounded half away from zero, nearest-neighbour replication back to full size).

Everything here is checked against numpy written from those two sentences, never against the oracle itself."""
import numpy as np
import pytest

import oracle as orc
from conftest import random_lf


def _ycocg_planes(lf):
    r, g, b = (lf[..., i].astype(np.int64) for i in range(3))
    co = r - b
    t = b + np.floor_divide(co, 2)
    cg = g - t
    y = t + np.floor_divide(cg, 2)
    return [y, co, cg]


def _box_down(p):
    """2 x 2 box mean, rounded half away from zero (integer arithmetic)."""
    s = p[..., 0::2, 0::2] + p[..., 0::2, 1::2] + p[..., 1::2, 0::2] + p[..., 1::2, 1::2]
    return np.sign(s) * ((2 * np.abs(s) + 4) // 8)


def _up(p):
    return np.repeat(np.repeat(p, 2, axis=-2), 2, axis=-1)


def _rgb_from(y, co, cg):
    t = y - np.floor_divide(cg, 2)
    g = cg + t
    b = t - np.floor_divide(co, 2)
    r = b + co
    return np.clip(np.stack([r, g, b], axis=-1), 0, 255).astype(np.uint8)


def _params(lf, h, B=4, W=4, tau_ref=0, tau_res=0, chroma=1, policy=orc.POLICY_ADAPTIVE):
    V, U, Ht, Ws, _ = lf.shape
    return orc.make_params(U, V, Ws, Ht, h, B, W, tau_ref, tau_res, policy, chroma=chroma)


def test_box_mean_worked_examples():
    # {1,1,3,3} -> 2; a constant plane stays constant; half away from zero on both sides
    assert _box_down(np.array([[1, 1], [3, 3]]))[0, 0] == 2
    assert _box_down(np.array([[1, 1], [1, 2]]))[0, 0] == 1      # 5/4 = 1.25
    assert _box_down(np.array([[1, 1], [2, 2]]))[0, 0] == 2      # 6/4 = 1.5 -> 2
    assert _box_down(np.array([[-1, -1], [-2, -2]]))[0, 0] == -2  # -1.5 -> -2
    # the oracle's level-0 chroma planes are exactly that filter of the full-resolution Co / Cg planes; luma is untouched
    rng = np.random.default_rng(11)
    lf = random_lf(rng, 3, 2, 16, 8, smooth=False)
    t = orc.Tree(lf, _params(lf, 1, W=1))
    X0 = _ycocg_planes(lf)
    for v in range(2):
        for u in range(3):
            assert np.array_equal(t.plane("X", 0, u, v, 0), X0[0][v, u])
            for c in (1, 2):
                got = t.plane("X", 0, u, v, c)
                assert got.shape == (4, 8)
                assert np.array_equal(got, _box_down(X0[c][v, u]))


def test_lossless_thresholds_give_the_closed_form():
    # tau = 0: nothing is dropped, so the decoder must return exactly clamp(inverse(Y, up(down(Co)), up(down(Cg)))) of the input;
    # P1 (encoder's reconstruction) = P2 (random access) = P3 (brute force) on every pixel
    rng = np.random.default_rng(12)
    lf = random_lf(rng, 4, 3, 16, 8)
    t = orc.Tree(lf, _params(lf, 2, W=3))
    y, co, cg = _ycocg_planes(lf)
    expect = _rgb_from(y, _up(_box_down(co)), _up(_box_down(cg)))
    assert np.array_equal(t.reconstruct(), expect)
    s = orc.Stream(t.serialize())
    assert np.array_equal(s.decode_full(), expect)
    coords = np.array([(u, v, x, yy) for v in range(3) for u in range(4) for yy in range(8) for x in range(16)], dtype=np.int32)
    assert np.array_equal(s.decode_brute(coords[::7]), expect[coords[::7, 1], coords[::7, 0], coords[::7, 3], coords[::7, 2]])
    assert s.params.chroma == 1


def test_grey_light_field_round_trips_exactly():
    # constant (zero) chroma survives the box mean: a grey light field is reproduced bit for bit at tau = 0
    rng = np.random.default_rng(13)
    g = rng.integers(0, 256, (2, 2, 8, 8, 1)).astype(np.uint8)
    lf = np.repeat(g, 3, axis=-1)
    t = orc.Tree(lf, _params(lf, 1, W=2))
    assert np.array_equal(orc.Stream(t.serialize()).decode_full(), lf)


@pytest.mark.parametrize("policy", [orc.POLICY_ADAPTIVE, orc.POLICY_ALL, orc.POLICY_LITERAL])
def test_lossy_p1_equals_p2_and_rate_drops(policy):
    rng = np.random.default_rng(14)
    lf = random_lf(rng, 4, 4, 32, 16)
    full = orc.Tree(lf, _params(lf, 2, W=4, tau_ref=20, tau_res=40, chroma=0, policy=policy))
    sub = orc.Tree(lf, _params(lf, 2, W=4, tau_ref=20, tau_res=40, chroma=1, policy=policy))
    b_full, b_sub = full.serialize(), sub.serialize()
    s = orc.Stream(b_sub)
    assert np.array_equal(s.decode_full(), sub.reconstruct())          # north_star pin 3 on the subsampled stream
    assert len(b_sub) < len(b_full)                                    # half-resolution chroma costs fewer bytes
    # the two losses separate: against the subsampled-but-unthresholded image (numpy closed form) only the thresholds are left,
    # and they cost about what they cost without subsampling
    y, co, cg = _ycocg_planes(lf)
    ideal = _rgb_from(y, _up(_box_down(co)), _up(_box_down(cg)))
    assert orc.psnr(ideal, sub.reconstruct()) > orc.psnr(lf, full.reconstruct()) - 3.0


def test_stream_sections_have_the_subsampled_sizes():
    # raw top-level RKVs: Y uint8 at Ws x Ht, Co / Cg int16 at Ws/2 x Ht/2; flag maps of chroma plane-channels
    # have ceil(nblk_c / 32) words
    rng = np.random.default_rng(15)
    lf = random_lf(rng, 2, 2, 16, 16)
    data = orc.Tree(lf, _params(lf, 1, W=2, tau_ref=10, tau_res=10)).serialize()
    assert data[49] == 1
    off_rkv, off_dir, off_flags, off_pay = (int.from_bytes(data[o:o + 8], "little") for o in (112, 120, 128, 136))
    n_top = 1
    assert off_dir - off_rkv == n_top * (16 * 16 + 2 * 2 * 8 * 8)
    # 1 reference plane (one map per channel) + 3 predictive planes (two maps); luma has 16 blocks, chroma 4: one 32-bit word per map;
    # sections are 8-byte aligned
    assert off_pay - off_flags == ((1 + 3 * 2) * 3 * 4 + 7) // 8 * 8


def test_geometry_that_does_not_divide_is_rejected():
    lf = np.zeros((1, 1, 12, 12, 3), dtype=np.uint8)   # 12 / 2 = 6 is not a multiple of B = 4
    with pytest.raises(orc.OracleError):
        orc.Tree(lf, _params(lf, 1, W=1))
    lf = np.zeros((1, 1, 8, 10, 3), dtype=np.uint8)    # 10 / 2 = 5
    with pytest.raises(orc.OracleError):
        orc.Tree(lf, _params(lf, 1, B=2, W=1))


def test_byte_counter_closed_form_with_subsampling():
    # every coordinate of a tau = 0 stream: each block of every plane-channel is touched once, chroma planes have a quarter of the blocks
    rng = np.random.default_rng(16)
    lf = random_lf(rng, 2, 2, 16, 8)
    s = orc.Stream(orc.Tree(lf, _params(lf, 1, W=2)).serialize())
    coords = np.array([(u, v, x, y) for v in range(2) for u in range(2) for y in range(8) for x in range(16)], dtype=np.int32)
    st = s.stats_decode(coords)
    nblk = [8, 2, 2]
    assert st["blocks_touched"] == 4 * sum(nblk)
    assert st["flag_bits"] == sum(nblk) * (1 + 3 * 2)
    assert st["rkv_bytes"] == 16 * 8 * 1 + 2 * (8 * 4) * 2
