"""Pins for the oracle's colour transform and BISE.

None of these re-type the oracle's formulas: they use hand-computed values, closed-form sizes,
information-theoretic bounds, exhaustive round trips, and a second, independently written
(sequential) decoder.
"""
import math

import numpy as np
import pytest

import oracle as orc


# ---------------------------------------------------------------- colour
def test_colour_exhaustive_roundtrip_and_ranges():
    # PAPER.md:263 "to avoid any loss of information due to transformations": all 2^24 triples
    assert orc.colour_roundtrip_failures() == 0


def test_colour_gray_maps_to_luma_only():
    # gray (g,g,g) -> (g,0,0)
    for g in (0, 1, 17, 128, 254, 255):
        assert orc.rgb_to_ycocg(g, g, g) == (g, 0, 0)


@pytest.mark.parametrize("rgb,ycc", [
    ((255, 0, 0), (63, 255, -127)),    # hand: co=255, t=0+127, cg=-127, y=127+floor(-127/2)=63
    ((0, 255, 0), (127, 0, 255)),      # co=0, t=0, cg=255, y=0+127
    ((0, 0, 255), (63, -255, -127)),   # co=-255, t=255+floor(-255/2)=255-128=127, cg=-127, y=127-64=63
    ((10, 20, 30), (20, -20, 0)),      # co=-20, t=30-10=20, cg=0, y=20
])
def test_colour_hand_values(rgb, ycc):
    assert orc.rgb_to_ycocg(*rgb) == ycc
    assert orc.ycocg_to_rgb(*ycc) == rgb


def test_colour_luma_is_close_to_weighted_mean():
    # YCoCg: Y ~ R/4 + G/2 + B/4 (the transform's definition up to the lifting floors)
    rng = np.random.default_rng(1)
    for r, g, b in rng.integers(0, 256, (500, 3)):
        y, co, cg = orc.rgb_to_ycocg(int(r), int(g), int(b))
        assert abs(y - (r / 4 + g / 2 + b / 4)) <= 1.0
        assert co == r - b


# ---------------------------------------------------------------- BISE layout choice and sizes
@pytest.mark.parametrize("N,layout,m,bits_per_15", [
    (1, orc.BISE_PLAIN, 0, 0),
    (2, orc.BISE_PLAIN, 1, 15),
    (3, orc.BISE_TRIT, 0, 24),          # 8 bits / 5 values = 1.6
    (5, orc.BISE_QUINT, 0, 35),         # 7 bits / 3 values = 2.33
    (8, orc.BISE_PLAIN, 3, 45),
    (33, orc.BISE_QUINT, 3, 80),        # 5*8 = 40 >= 33 : 7/3 + 3 = 5.33
    (80, orc.BISE_QUINT, 4, 95),        # 5*16 = 80 : 6.33
    (223, orc.BISE_PLAIN, 8, 120),      # trit m=7 (384): 8.6, quint m=6 (320): 8.33, plain 8 wins
    (2041, orc.BISE_PLAIN, 11, 165),
    (2178, orc.BISE_QUINT, 9, 170),     # MV records, W=16: 11.33 bits
])
def test_bise_choose_closed_forms(N, layout, m, bits_per_15):
    assert orc.bise_choose(N) == (layout, m)
    assert orc.bise_nbits(N, 15) == bits_per_15


def test_bise_never_worse_than_plain_and_never_below_entropy():
    for N in list(range(1, 300)) + [511, 512, 513, 1000, 2041, 2178, 40000, 65536]:
        bits15 = orc.bise_nbits(N, 15)
        plain = 15 * (0 if N <= 1 else math.ceil(math.log2(N)))
        assert bits15 <= plain
        assert bits15 >= 15 * math.log2(N) - 1e-9      # cannot beat log2 N bits/value
        assert bits15 <= 15 * math.log2(max(N, 2)) + 15  # within one bit/value of the bound


def test_bise_golden_bits():
    # trit group: T = sum t_k 3^k ; [0,1,2,0,1] -> 0 + 3 + 18 + 0 + 81 = 102
    assert orc.bise_encode([0, 1, 2, 0, 1], 3)[0] == 102
    # quint group: Q = sum q_k 5^k ; [4,0,3] -> 4 + 0 + 75 = 79 (7 bits)
    assert orc.bise_encode([4, 0, 3], 5)[0] == 79
    # N=6: trit m=1, value = t*2 + low. [5,0,3,2,4] -> t=[2,0,1,1,2], low=[1,0,1,0,0]
    # T = 2 + 0 + 9 + 27 + 162 = 200 -> byte0 = 200 ; lows LSB-first in bits 8..12 = 0b00101 = 5
    bits = orc.bise_encode([5, 0, 3, 2, 4], 6)
    assert (bits[0], bits[1]) == (200, 5)
    # plain, N=8, 3 bits LSB-first: [7,1,2] -> 0b010_001_111 = 0x8F, 0x00
    bits = orc.bise_encode([7, 1, 2], 8)
    assert (bits[0], bits[1]) == (0x8F, 0x00)


@pytest.mark.parametrize("N", [1, 2, 3, 5, 6, 8, 10, 17, 33, 80, 223, 255, 2041, 2178, 65536])
def test_bise_roundtrip_random_access_and_sequential(N):
    rng = np.random.default_rng(N)
    count = 1003
    vals = rng.integers(0, N, count).astype(np.uint32)
    bits = orc.bise_encode(vals, N)
    assert bits.size >= orc.bise_nbits(N, count) // 8
    seq = orc.bise_decode_seq(bits, N, count)
    assert np.array_equal(seq, vals)
    for i in rng.permutation(count)[:400]:
        assert orc.bise_decode_at(bits, N, int(i)) == vals[i]


def test_bise_many_ranges_roundtrip():
    rng = np.random.default_rng(7)
    for N in rng.integers(1, 2 ** 16 + 1, 60):
        N = int(N)
        vals = rng.integers(0, N, 97).astype(np.uint32)
        bits = orc.bise_encode(vals, N)
        assert np.array_equal(orc.bise_decode_seq(bits, N, 97), vals)
        assert all(orc.bise_decode_at(bits, N, i) == vals[i] for i in (0, 1, 48, 95, 96))


def test_bise_rejects_out_of_range():
    with pytest.raises(orc.OracleError):
        orc.bise_encode([0, 3], 3)
