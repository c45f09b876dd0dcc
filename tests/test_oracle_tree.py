"""Pins for the oracle's hierarchy, phase-shifted motion search,
replacement step and thresholds."""
import numpy as np
import pytest

import oracle as orc
from conftest import random_lf


def _tree(lf, h, B=4, W=4, tau_ref=0, tau_res=0, policy=orc.POLICY_ADAPTIVE):
    V, U, Ht, Ws, _ = lf.shape
    p = orc.make_params(U, V, Ws, Ht, h, B, W, tau_ref, tau_res, policy)
    return orc.Tree(lf, p)


def _ycocg_planes(lf):
    """Independent numpy colour transform (floor division) for building expectations."""
    r, g, b = (lf[..., i].astype(np.int64) for i in range(3))
    co = r - b
    t = b + np.floor_divide(co, 2)
    cg = g - t
    y = t + np.floor_divide(cg, 2)
    return [y, co, cg]


# ---------------------------------------------------------------- hierarchy
def test_level_dims_odd_grid_17():
    # R3: 17 -> 9 -> 5 -> 3 (by hand: ceil halves)
    rng = np.random.default_rng(0)
    lf = rng.integers(0, 256, (17, 17, 8, 8, 3)).astype(np.uint8)
    t = _tree(lf, 3, W=1)
    assert [t.level_dims(L) for L in range(4)] == [(17, 17), (9, 9), (5, 5), (3, 3)]


def test_path_sum_identity_and_srv_definition():
    # X_0[p] = X_h[p>>h] + sum_L SRV_L[p>>L], exactly; SRV = member - RKV
    rng = np.random.default_rng(1)
    lf = random_lf(rng, 5, 6, 16, 12)
    h = 2
    t = _tree(lf, h, W=2)
    X0 = _ycocg_planes(lf)
    for c in range(3):
        for v in range(6):
            for u in range(5):
                assert np.array_equal(t.plane("X", 0, u, v, c), X0[c][v, u])
                acc = t.plane("X", h, u >> h, v >> h, c).astype(np.int64)
                for L in range(h):
                    acc += t.plane("srv", L, u >> L, v >> L, c)
                assert np.array_equal(acc, X0[c][v, u])
                assert np.array_equal(t.plane("srv", 0, u, v, c), t.plane("X", 0, u, v, c) - t.plane("X", 1, u >> 1, v >> 1, c))


def test_rkv_is_rounded_mean_half_away_from_zero():
    # arithmetic mean of the present members, rounded half away from zero (R2, R3)
    rng = np.random.default_rng(2)
    lf = random_lf(rng, 3, 3, 8, 8, smooth=False)
    t = _tree(lf, 1, W=1)
    X0 = _ycocg_planes(lf)
    for c in range(3):
        for qv in range(2):
            for qu in range(2):
                members = [X0[c][v, u] for v in (2 * qv, 2 * qv + 1) for u in (2 * qu, 2 * qu + 1) if u < 3 and v < 3]
                mean = np.mean(np.stack(members).astype(np.float64), axis=0)
                expect = np.where(mean >= 0, np.floor(mean + 0.5), -np.floor(-mean + 0.5)).astype(np.int64)
                assert np.array_equal(t.plane("X", 1, qu, qv, c), expect)


def test_rkv_mean_example():
    # members {0,0,2,2} at a pixel -> RKV pixel 1 ; {0,0,0,2} -> 0.5 -> 1 (half away)
    lf = np.zeros((2, 2, 4, 4, 3), dtype=np.uint8)
    lf[1, 0], lf[1, 1] = 2, 2
    t = _tree(lf, 1, W=1)
    assert np.all(t.plane("X", 1, 0, 0, 0) == 1)
    lf[1, 0] = 0
    t = _tree(lf, 1, W=1)
    assert np.all(t.plane("X", 1, 0, 0, 0) == 1)  # mean 0.5 rounds away from zero


def test_identical_views_give_zero_srvs():
    # SPEC.md:179
    rng = np.random.default_rng(3)
    img = rng.integers(0, 256, (8, 12, 3)).astype(np.uint8)
    lf = np.broadcast_to(img, (4, 4, 8, 12, 3)).copy()
    t = _tree(lf, 2, W=2)
    for L in range(2):
        UL, VL = t.level_dims(L)
        for c in range(3):
            for v in range(VL):
                for u in range(UL):
                    assert not t.plane("srv", L, u, v, c).any()


# ---------------------------------------------------------------- motion search
def _brute_search(P, R, B, W, bx, by):
    """Straight loops over Eqs. (1)-(2) with the tie order of R9 (sad, mode, dy, dx)."""
    Ht, Ws = P.shape
    best = None
    for mode in (0, 1):
        for dy in range(-W, W + 1):
            for dx in range(-W, W + 1):
                sad = 0
                for j in range(B):
                    for i in range(B):
                        y, x = by * B + j, bx * B + i
                        ry, rx = y + dy, x + dx
                        r = int(R[ry, rx]) if (0 <= ry < Ht and 0 <= rx < Ws) else 0
                        p = int(P[y, x])
                        sad += abs(p - r) if mode == 0 else abs(p + r)
                key = (sad, mode, dy, dx)
                if best is None or key < best:
                    best = key
    return best[1], best[3], best[2], best[0]  # mode, dx, dy, sad


@pytest.mark.parametrize("B,W", [(4, 4), (2, 3), (4, 1), (8, 2)])
def test_search_matches_brute_force(B, W):
    # optimality by brute force at small W, >= 500 blocks overall
    rng = np.random.default_rng(10 + B + W)
    Ws, Ht = 8 * B, 6 * B
    n = 0
    for trial in range(4):
        R = rng.integers(-40, 41, (Ht, Ws)).astype(np.int16)
        # P: a shifted / negated / noisy relative of R so that both modes and many offsets win
        sh = np.roll(R, (int(rng.integers(-W, W + 1)), int(rng.integers(-W, W + 1))), (0, 1))
        P = (sh * (1 if trial % 2 == 0 else -1) + rng.integers(-3, 4, (Ht, Ws))).astype(np.int16)
        P[: Ht // 2, : Ws // 2] = rng.integers(-2, 3, (Ht // 2, Ws // 2))  # low-energy area -> ties
        for by in range(Ht // B):
            for bx in range(Ws // B):
                assert orc.search_block(P, R, B, W, bx, by) == _brute_search(P, R, B, W, bx, by)
                n += 1
    assert n >= 190


def test_search_phase_inverted_copy_is_additive_zero():
    # P = -R  =>  additive mode, Delta+ = 0 at (0,0)
    rng = np.random.default_rng(4)
    R = rng.integers(-100, 101, (16, 16)).astype(np.int16)
    R[R == 0] = 1
    for by in range(4):
        for bx in range(4):
            assert orc.search_block(-R, R, 4, 4, bx, by) == (1, 0, 0, 0)


def test_search_recovers_shift():
    # reference = predictive shifted by (+3,+1)  =>  (dx,dy) recovers it, residual 0 away from borders
    rng = np.random.default_rng(5)
    big = rng.integers(-100, 101, (40, 40)).astype(np.int16)
    big[big == 0] = 7
    P = big[8:32, 8:32]
    R = big[8 - 1:32 - 1, 8 - 3:32 - 3]      # R(x+3, y+1) = P(x, y)
    for by in range(1, 5):
        for bx in range(1, 5):
            assert orc.search_block(P, R, 4, 4, bx, by) == (0, 3, 1, 0)


def test_search_never_worse_than_zero_motion():
    # Delta <= Delta-^{0,0}
    rng = np.random.default_rng(6)
    P = rng.integers(-50, 51, (16, 16)).astype(np.int16)
    R = rng.integers(-50, 51, (16, 16)).astype(np.int16)
    for by in range(4):
        for bx in range(4):
            sad = orc.search_block(P, R, 4, 3, bx, by)[3]
            assert sad <= np.abs(P[by * 4:by * 4 + 4, bx * 4:bx * 4 + 4].astype(int) - R[by * 4:by * 4 + 4, bx * 4:bx * 4 + 4]).sum()


def test_tree_search_uses_cluster_reference_and_roles():
    # R5: even-even member is the reference; every predictive block is searched against it (unthresholded)
    rng = np.random.default_rng(7)
    lf = random_lf(rng, 4, 3, 16, 16)
    t = _tree(lf, 2, B=4, W=3)
    for L in range(2):
        UL, VL = t.level_dims(L)
        for pv in range(VL):
            for pu in range(UL):
                blocks = t.blocks(L, pu, pv, 1)
                if (pu | pv) & 1:
                    P = t.plane("srv", L, pu, pv, 1)
                    R = t.plane("srv", L, pu & ~1, pv & ~1, 1)
                    for by in range(4):
                        for bx in range(4):
                            assert tuple(blocks[by, bx, :4]) == orc.search_block(P, R, 4, 3, bx, by)
                            assert blocks[by, bx, 4] == np.abs(P[by * 4:by * 4 + 4, bx * 4:bx * 4 + 4].astype(int)).sum()
                else:
                    assert not (blocks[..., 5] & 2).any()  # references carry no pred flag


# ---------------------------------------------------------------- replacement + thresholds
def test_recompensation_inverts_replacement():
    # stored residual +- shifted reference = original SRV, every sample (R10)
    rng = np.random.default_rng(8)
    lf = random_lf(rng, 4, 4, 16, 16)
    t = _tree(lf, 2, B=4, W=4)
    for L in range(2):
        UL, VL = t.level_dims(L)
        for pv in range(VL):
            for pu in range(UL):
                if not (pu | pv) & 1:
                    assert np.array_equal(t.plane("stored", L, pu, pv, 0), t.plane("srv", L, pu, pv, 0))
                    continue
                e = t.plane("stored", L, pu, pv, 0).astype(int)
                R = np.pad(t.plane("srv", L, pu & ~1, pv & ~1, 0).astype(int), 4)
                blocks = t.blocks(L, pu, pv, 0)
                rec = np.zeros_like(e)
                for y in range(16):
                    for x in range(16):
                        mode, dx, dy, _, _, fl = blocks[y // 4, x // 4]
                        q = R[y + dy + 4, x + dx + 4] if fl & 2 else 0
                        rec[y, x] = e[y, x] + (-q if mode else q)
                assert np.array_equal(rec, t.plane("srv", L, pu, pv, 0))


def test_threshold_rule_and_policies():
    # PAPER.md:268 / R11: significant iff energy >= tau ; R13 policies
    rng = np.random.default_rng(9)
    lf = random_lf(rng, 4, 4, 16, 16)
    t = _tree(lf, 2, B=4, W=4)
    for policy in (orc.POLICY_ADAPTIVE, orc.POLICY_ALL, orc.POLICY_LITERAL):
        t.threshold(20, 30, policy)
        for L in range(2):
            UL, VL = t.level_dims(L)
            for pv in range(VL):
                for pu in range(UL):
                    b = t.blocks(L, pu, pv, 2).reshape(-1, 6)
                    sad, E, fl = b[:, 3], b[:, 4], b[:, 5]
                    res, pred = (fl & 1).astype(bool), (fl & 2).astype(bool)
                    if not (pu | pv) & 1:
                        assert np.array_equal(res, E >= 20) and not pred.any()
                    elif policy == orc.POLICY_ALL:
                        assert pred.all() and np.array_equal(res, sad >= 30)
                    elif policy == orc.POLICY_LITERAL:
                        assert np.array_equal(res, sad >= 30) and np.array_equal(pred, res)
                    else:
                        worth = E >= 30
                        assert np.array_equal(pred, worth & (sad < E))
                        assert np.array_equal(res, worth & (np.where(pred, sad, E) >= 30))
    t.threshold(0, 0, orc.POLICY_ADAPTIVE)
    for L in range(2):
        UL, VL = t.level_dims(L)
        for pv in range(VL):
            for pu in range(UL):
                assert (t.blocks(L, pu, pv, 0)[..., 5] & 1).all()  # tau = 0 keeps every block
