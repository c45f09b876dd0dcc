"""Pins for the oracle's half-pel motion compensation (section 6: "sub-pel motion compensation, i.e., sub-pixel level
motion compensation to search for a matching block using bi-linear interpolation methods"; R28: offsets in half pixels,
range [-2W, 2W]^2, reference value = mean of the 1 / 2 / 4 integer samples around the position, rounded half up, 0 outside the image).

Everything here is checked against numpy written from that sentence, never against the oracle itself."""
import numpy as np
import pytest

import oracle as orc
from conftest import random_lf


def _interp(R, x2, y2):
    """Bilinear value of plane R at the half-pel position (x2 / 2, y2 / 2), integer arithmetic, zeros outside."""
    H, W = R.shape

    def at(x, y):
        return int(R[y, x]) if 0 <= x < W and 0 <= y < H else 0

    x0, y0 = x2 // 2, y2 // 2          # Python's // is floor
    fx, fy = x2 - 2 * x0, y2 - 2 * y0
    pts = [(x0, y0)] + ([(x0 + 1, y0)] if fx else []) + ([(x0, y0 + 1)] if fy else []) + ([(x0 + 1, y0 + 1)] if fx and fy else [])
    s, n = sum(at(x, y) for x, y in pts), len(pts)
    return s if n == 1 else (s + n // 2) // n


def _sad(P, R, B, bx, by, dx2, dy2, mode):
    tot = 0
    for j in range(B):
        for i in range(B):
            x, y = bx * B + i, by * B + j
            r = _interp(R, 2 * x + dx2, 2 * y + dy2)
            tot += abs(int(P[y, x]) + r) if mode else abs(int(P[y, x]) - r)
    return tot


def _brute(P, R, B, W, bx, by):
    """Exhaustive search written from Eqs. (1)-(2) on the half-pel grid; ties: subtractive first, then smallest dy, then dx (R9)."""
    best = None
    for mode in (0, 1):
        for dy in range(-2 * W, 2 * W + 1):
            for dx in range(-2 * W, 2 * W + 1):
                s = _sad(P, R, B, bx, by, dx, dy, mode)
                if best is None or s < best[3]:
                    best = (mode, dx, dy, s)
    return best


def test_rounding_worked_examples():
    # 2 samples: (a + b + 1) >> 1 with floor for negative sums; 4 samples: (a + b + c + d + 2) >> 2
    R = np.array([[1, 2], [4, 8]], dtype=np.int16)
    assert _interp(R, 1, 0) == 2      # (1 + 2 + 1) // 2
    assert _interp(R, 0, 1) == 3      # (1 + 4 + 1) // 2
    assert _interp(R, 1, 1) == 4      # (15 + 2) // 4
    assert _interp(-R, 1, 0) == -1    # (-3 + 1) // 2 = -1: half up, not away from zero
    assert _interp(R, 3, 0) == 1      # (2 + 0 + 1) // 2: the sample right of the image reads 0
    assert _interp(R, -1, -1) == 0    # (0 + 0 + 0 + 1 + 2) // 4
    # the oracle's search reproduces them: a block that IS the interpolated reference is found with Delta = 0 at that offset
    rng = np.random.default_rng(3)
    R = rng.integers(-200, 200, (16, 16)).astype(np.int16)
    for dx2, dy2 in ((3, 0), (0, -3), (1, 1), (-5, 3), (4, 2)):
        P = np.array([[_interp(R, 2 * x + dx2, 2 * y + dy2) for x in range(16)] for y in range(16)], dtype=np.int16)
        assert orc.search_block_halfpel(P, R, 4, 4, 1, 2) == (0, dx2, dy2, 0)
        assert orc.search_block_halfpel(-P, R, 4, 4, 1, 2) == (1, dx2, dy2, 0)   # the sign-inverted block: additive mode (R10)


@pytest.mark.parametrize("B,W", [(4, 2), (2, 3), (8, 1)])
def test_search_equals_brute_force_and_never_loses_to_integer_pel(B, W):
    rng = np.random.default_rng(100 + B)
    P = rng.integers(-60, 60, (2 * B, 3 * B)).astype(np.int16)
    R = (P + rng.integers(-8, 8, P.shape)).astype(np.int16)
    R = np.roll(R, (1, -1), axis=(0, 1))
    for by in range(2):
        for bx in range(3):
            got = orc.search_block_halfpel(P, R, B, W, bx, by)
            assert got == _brute(P, R, B, W, bx, by)
            assert got[3] <= orc.search_block(P, R, B, W, bx, by)[3]   # the even offsets are the integer-pel candidates


def _params(lf, h, B=4, W=3, tau_ref=0, tau_res=0, subpel=1, policy=orc.POLICY_ADAPTIVE, chroma=0):
    V, U, Ht, Ws, _ = lf.shape
    return orc.make_params(U, V, Ws, Ht, h, B, W, tau_ref, tau_res, policy, subpel=subpel, chroma=chroma)


@pytest.mark.parametrize("policy", [orc.POLICY_ADAPTIVE, orc.POLICY_ALL, orc.POLICY_LITERAL])
def test_p1_p2_p3_agree_and_lossless_round_trip(policy):
    rng = np.random.default_rng(21)
    lf = random_lf(rng, 4, 3, 16, 8)
    t = orc.Tree(lf, _params(lf, 2, policy=policy))
    s = orc.Stream(t.serialize())
    assert s.params.subpel == 1
    assert np.array_equal(t.reconstruct(), lf)          # tau = 0: nothing dropped, the input comes back
    assert np.array_equal(s.decode_full(), lf)
    coords = np.array([(u, v, x, y) for v in range(3) for u in range(4) for y in range(8) for x in range(16)], dtype=np.int32)[::3]
    assert np.array_equal(s.decode_brute(coords), lf[coords[:, 1], coords[:, 0], coords[:, 3], coords[:, 2]])
    lossy = orc.Tree(lf, _params(lf, 2, tau_ref=15, tau_res=30, policy=policy))
    sl = orc.Stream(lossy.serialize())
    assert np.array_equal(sl.decode_full(), lossy.reconstruct())   # north_star pin 3 on the half-pel stream
    assert np.array_equal(sl.decode_brute(coords), lossy.reconstruct()[coords[:, 1], coords[:, 0], coords[:, 3], coords[:, 2]])


def test_offsets_are_stored_in_half_pixels_and_the_flag_is_in_the_header():
    rng = np.random.default_rng(22)
    lf = random_lf(rng, 2, 2, 16, 8)
    W = 2
    t = orc.Tree(lf, _params(lf, 1, W=W, tau_res=1, policy=orc.POLICY_ALL))
    data = t.serialize()
    assert data[55] == 1
    assert orc.Tree(lf, _params(lf, 1, W=W, subpel=0)).serialize()[55] == 0
    blocks = t.blocks(0, 1, 0, 0).reshape(-1, 6)   # a predictive plane: mode, dx, dy, sad, E, flags per block (row-major)
    assert np.abs(blocks[:, 1:3]).max() <= 2 * W and (np.abs(blocks[:, 1:3]) % 2 == 1).any()   # odd = true half-pel offsets occur
    # each block's Delta is the numpy SAD at its stored offset
    P, R = t.plane("srv", 0, 1, 0, 0), t.plane("srv", 0, 0, 0, 0)
    nbx = 16 // 4
    for b, (mode, dx, dy, sad, *_rest) in enumerate(blocks):
        assert sad == _sad(P, R, 4, b % nbx, b // nbx, int(dx), int(dy), int(mode))


def test_half_pixel_shift_is_predicted_better():
    # a plane that is its reference moved by half a pixel (plus a little noise): Delta of every block can only fall against the
    # integer-pel search (candidate superset) and falls strictly in total
    rng = np.random.default_rng(23)
    base = rng.integers(-120, 120, (16, 40)).astype(np.float64)
    base = (base + np.roll(base, 1, 1) + np.roll(base, 2, 1) + np.roll(base, 1, 0)) / 4.0   # smooth enough to interpolate
    R = np.rint(base[:, 4:36]).astype(np.int16)
    P = np.rint(0.5 * (base[:, 5:37] + base[:, 6:38]) + rng.normal(0, 0.5, (16, 32))).astype(np.int16)   # R moved by 1.5 pixels
    tot_i = tot_h = 0
    for by in range(4):
        for bx in range(1, 7):
            si, sh = orc.search_block(P, R, 4, 2, bx, by)[3], orc.search_block_halfpel(P, R, 4, 2, bx, by)[3]
            assert sh <= si
            tot_i += si; tot_h += sh
    assert tot_h < 0.7 * tot_i


def test_byte_counter_closed_form_with_half_pel():
    # every coordinate of a tau = 0 stream: each block of every plane-channel is touched once however many reference samples a tap blends
    rng = np.random.default_rng(24)
    lf = random_lf(rng, 2, 2, 16, 8)
    s = orc.Stream(orc.Tree(lf, _params(lf, 1, W=2)).serialize())
    coords = np.array([(u, v, x, y) for v in range(2) for u in range(2) for y in range(8) for x in range(16)], dtype=np.int32)
    st = s.stats_decode(coords)
    nblk = 8
    assert st["blocks_touched"] == 4 * 3 * nblk
    assert st["flag_bits"] == 3 * nblk * (1 + 3 * 2)


def test_combines_with_chroma_subsampling():
    rng = np.random.default_rng(25)
    lf = random_lf(rng, 2, 2, 16, 16)
    t = orc.Tree(lf, _params(lf, 1, W=2, tau_ref=8, tau_res=16, chroma=1))
    s = orc.Stream(t.serialize())
    assert s.params.subpel == 1 and s.params.chroma == 1
    assert np.array_equal(s.decode_full(), t.reconstruct())
