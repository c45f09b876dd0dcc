"""GPU parity of hmlfc_search (phase-shifted exhaustive block motion search, Eqs. 1-2) against the
oracle's search, block by block, bit-exact: mode, motion vector and minimum SAD including every tie."""
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


def _oracle_all_blocks(Pp, Rp, B, W):
    Ht, Ws = Pp.shape
    out = np.empty((Ht // B, Ws // B, 4), dtype=np.int32)
    for by in range(Ht // B):
        for bx in range(Ws // B):
            out[by, bx] = orc.search_block(Pp, Rp, B, W, bx, by)
    return out


def _gpu(P, planes, pairs, B, W):
    d = P.hmlfc_search(torch.from_numpy(np.ascontiguousarray(planes)).cuda(),
                       torch.from_numpy(np.ascontiguousarray(pairs, dtype=np.int32)).cuda(), B, W)
    torch.cuda.synchronize()
    return d.cpu().numpy()


@pytest.mark.parametrize("Ws,Ht,B,W", [(40, 24, 4, 1), (40, 24, 4, 3), (36, 20, 4, 16), (64, 32, 4, 16), (8, 8, 4, 16),
                                        (4, 4, 4, 2), (44, 12, 4, 33), (20, 12, 2, 5), (32, 16, 8, 6), (12, 12, 1, 2)])
def test_search_matches_oracle_on_random_planes(P, Ws, Ht, B, W):
    rng = np.random.default_rng(Ws * 1000 + Ht * 10 + W)
    # smooth-ish signed planes with coherent shifted / inverted copies, like SRV images
    base = rng.integers(-200, 201, (Ht + 2 * 8, Ws + 2 * 8)).astype(np.int16)
    R = base[8:8 + Ht, 8:8 + Ws].copy()
    P1 = (base[8 + 1:8 + 1 + Ht, 8 - 2:8 - 2 + Ws] + rng.integers(-3, 4, (Ht, Ws))).astype(np.int16)   # shifted copy + noise
    P2 = (-base[8 - 1:8 - 1 + Ht, 8 + 1:8 + 1 + Ws]).astype(np.int16)                                  # phase-inverted shifted copy
    P3 = rng.integers(-510, 511, (Ht, Ws)).astype(np.int16)                                            # unrelated
    planes = np.stack([R, P1, P2, P3])
    pairs = np.array([[1, 0], [2, 0], [3, 0], [0, 0]], dtype=np.int32)
    got = _gpu(P, planes, pairs, B, W)
    for k, (p, r) in enumerate(pairs):
        assert np.array_equal(got[k], _oracle_all_blocks(planes[p], planes[r], B, W)), (k, Ws, Ht, B, W)
    if B >= 4 and W >= 2 and min(Ws, Ht) > 2 * B + 4:
        inner = got[1][1:-1, 1:-1]                       # interior blocks of the inverted copy: additive, exact
        assert (inner[..., 0] == 1).all() and (inner[..., 3] == 0).all()
        assert (inner[..., 1] == 1).all() and (inner[..., 2] == -1).all()


def test_search_ties_and_extreme_values(P):
    Ws, Ht, B, W = 32, 16, 4, 16
    zeros = np.zeros((Ht, Ws), np.int16)
    big = np.full((Ht, Ws), 32767, np.int16)
    neg = np.full((Ht, Ws), -32768, np.int16)
    planes = np.stack([zeros, big, neg])
    pairs = np.array([[0, 0], [1, 2], [2, 1], [1, 1]], dtype=np.int32)
    got = _gpu(P, planes, pairs, B, W)
    # all-zero planes: every offset ties at 0 -> subtractive, smallest dy, then smallest dx (R9)
    assert (got[0] == np.array([0, -W, -W, 0])).all()
    for k, (p, r) in enumerate(pairs):
        assert np.array_equal(got[k], _oracle_all_blocks(planes[p], planes[r], B, W)), k


@pytest.mark.parametrize("name", ["mini2", "mini4"])
def test_search_reproduces_the_encoders_decisions_on_real_srv_planes(P, name):
    """All predictive planes of every level and channel of an encoded light field: the GPU search on the oracle's SRV
    images gives the (mode, dx, dy, SAD) the oracle encoder stored for every block."""
    cfg = wl.CONFIGS[name]
    lf = wl.light_field(cfg)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, cfg.tau_res // 2, cfg.tau_res,
                        geometry=wl.geometry(cfg), seed=cfg.seed)
    tree = orc.Tree(lf, p)
    n_checked = 0
    for L in range(cfg.height):
        UL, VL = tree.level_dims(L)
        for c in range(3):
            planes = np.stack([tree.plane("srv", L, pu, pv, c) for pv in range(VL) for pu in range(UL)])
            pairs = [(pv * UL + pu, (pv & ~1) * UL + (pu & ~1)) for pv in range(VL) for pu in range(UL) if (pu | pv) & 1]
            got = _gpu(P, planes, np.array(pairs, dtype=np.int32), cfg.block, cfg.window)
            for k, (pi, ri) in enumerate(pairs):
                expect = tree.blocks(L, pi % UL, pi // UL, c)[..., :4]
                assert np.array_equal(got[k], expect), (L, c, pi)
                n_checked += expect.shape[0] * expect.shape[1]
    tree.close()
    assert n_checked > 10_000
