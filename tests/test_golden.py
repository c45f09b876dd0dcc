"""The oracle against the fixtures in tests/golden/ (values the paper prints, or worked by hand from its formulas)."""
import os

import numpy as np
import pytest

import oracle as orc

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _rows(name):
    with open(os.path.join(GOLDEN, name)) as fh:
        return [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]


def test_table1_sizes_and_ratio_range_fix_the_rate_definitions():
    """PAPER.md:323-329.  'Size (MB)' = U*V*W*H*3 bytes / 2^20 for 24-bit RGB, and 24 bpp / rate reproduces the abstract's
    30-800x: so rate = total bits / light-field PIXELS (not samples) -- the definition the oracle's `bpp` uses."""
    rows = _rows("table1_datasets.txt")
    assert len(rows) == 7
    ratios = []
    for name, U, V, W, H, mb, bpp, psnr in rows:
        U, V, W, H, mb, bpp, psnr = int(U), int(V), int(W), int(H), int(mb), float(bpp), float(psnr)
        assert U * V * W * H * 3 == mb << 20, name
        assert 40.0 <= psnr <= 45.0
        ratios.append(24.0 / bpp)
    assert 30.0 <= min(ratios) < 40.0 and 800.0 <= max(ratios) < 900.0   # "30-800x"
    # the oracle reports the same quantity: 8 * stream bytes / (U V Ws Ht)
    rng = np.random.default_rng(5)
    lf = rng.integers(0, 256, (2, 2, 8, 8, 3), dtype=np.uint8)
    data, info, tree = orc.encode(lf, orc.make_params(2, 2, 8, 8, 1, 4, 2))
    tree.close()
    assert info["bpp"] == 8.0 * len(data) / (2 * 2 * 8 * 8) and info["stream_bytes"] == len(data)


def test_eq12_worked_block():
    """every offset's SAD pair of the hand-worked block, the minimum, and the residual."""
    R = np.array([[1, -2, 3, 0], [4, 5, -6, 7], [-8, 9, 10, -11], [12, -13, 14, 15]], dtype=np.int16)
    P = np.zeros((4, 4), dtype=np.int16)
    P[2:, 2:] = [[-9, -10], [13, -14]]
    rows = _rows("eq12_worked_block.txt")
    per_offset = [tuple(int(x) for x in r) for r in rows if len(r) == 4 and r[0] != "best"]
    assert len(per_offset) == 9
    for dx, dy, dm, dp in per_offset:
        # shift the reference by hand (zero outside the image, R8), then ask the oracle for the zero-window search
        Rs = np.zeros_like(R)
        for y in range(4):
            for x in range(4):
                if 0 <= x + dx < 4 and 0 <= y + dy < 4:
                    Rs[y, x] = R[y + dy, x + dx]
        mode, mx, my, sad = orc.search_block(P, Rs, 2, 0, 1, 1)
        assert (mx, my) == (0, 0) and sad == min(dm, dp), (dx, dy)
        assert mode == (1 if dp < dm else 0)                          # ties: subtractive first (R9)
    best = [r for r in rows if r[0] == "best"][0]
    mode, dx, dy, sad = orc.search_block(P, R, 2, 1, 1, 1)
    assert (("additive" if mode else "subtractive"), dx, dy, sad) == (best[1], int(best[2]), int(best[3]), int(best[4]))
    assert sad == min(min(dm, dp) for _, _, dm, dp in per_offset)
    # the residual, through the encoder itself: a gray 2 x 2 light field whose Y planes are 128 + R, 128 + P, 128 - R,
    # 128 - P has the cluster mean 128 everywhere, so its level-0 SRV images are exactly R (reference, view (0,0)) and P (view (1,0))
    for tag, Pk in (("", P), ("2", P + np.array([[0, 0, 0, 0], [0, 0, 0, 0], [0, 0, 0, 0], [0, 0, 0, 1]], dtype=np.int16))):
        planes = [128 + R, 128 + Pk, 128 - R, 128 - Pk]   # views (u,v) = (0,0), (1,0), (0,1), (1,1)
        lf = np.stack([np.repeat(p.astype(np.uint8)[..., None], 3, axis=-1) for p in planes]).reshape(2, 2, 4, 4, 3)
        tree = orc.Tree(lf, orc.make_params(2, 2, 4, 4, 1, 2, 1, 0, 0, policy=orc.POLICY_ALL))
        assert np.array_equal(tree.plane("srv", 0, 0, 0, 0), R) and np.array_equal(tree.plane("srv", 0, 1, 0, 0), Pk)
        tree.threshold(0, 0)
        bestk = [r for r in rows if r[0] == "best" + tag][0]
        mode, dx, dy, sad = tree.blocks(0, 1, 0, 0)[1, 1, :4]
        assert (("additive" if mode else "subtractive"), dx, dy, sad) == (bestk[1], int(bestk[2]), int(bestk[3]), int(bestk[4]))
        resid = [int(x) for x in [r for r in rows if r[0] == "residual" + tag][0][1:]]
        assert tree.plane("stored", 0, 1, 0, 0)[2:, 2:].ravel().tolist() == resid
        tree.close()


def test_bise_groups_and_sizes():
    """group bit patterns and bits per value."""
    for row in _rows("bise_groups.txt"):
        if row[0] == "group":
            N, vals, expect = int(row[1]), [int(v) for v in row[2].split(",")], [int(v) for v in row[3].split(",")]
            bits = orc.bise_encode(vals, N)
            assert list(bits[:len(expect)]) == expect, row
            assert [orc.bise_decode_at(bits, N, i) for i in range(len(vals))] == vals
        else:
            N, layout, m, bits15 = (int(v) for v in row[1:])
            assert orc.bise_choose(N) == (layout, m), row
            assert orc.bise_nbits(N, 15) == bits15, row


def test_ycocg_hand_values():
    """PAPER.md:263."""
    for r, g, b, y, co, cg in ((int(v) for v in row) for row in _rows("ycocg_hand_values.txt")):
        assert orc.rgb_to_ycocg(r, g, b) == (y, co, cg)
        assert orc.ycocg_to_rgb(y, co, cg) == (r, g, b)
