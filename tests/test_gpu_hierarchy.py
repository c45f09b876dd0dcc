"""GPU parity of hmlfc_hierarchy (forward YCoCg-R + RLFC hierarchy build) against the oracle's encoder:
every SRV plane of every level and the top-level RKVs, bit-exact; then search + hierarchy together reproduce the oracle
encoder's motion decisions from the RGB light field alone."""
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


def _tree(cfg, lf):
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, cfg.tau_res // 2, cfg.tau_res,
                        geometry=wl.geometry(cfg), seed=cfg.seed)
    return orc.Tree(lf, p)


@pytest.mark.parametrize("name", ["cfg1", "mini2", "mini3", "mini4"])   # mini3: odd 5 x 5 grid (partial clusters, R3)
def test_hierarchy_matches_the_oracle_tree(P, name):
    cfg = wl.CONFIGS[name]
    lf = wl.light_field(cfg)
    tree = _tree(cfg, lf)
    srv, x = P.hmlfc_hierarchy(torch.from_numpy(lf).cuda(), cfg.height)
    torch.cuda.synchronize()
    srv, x = srv.cpu().numpy(), x.cpu().numpy()
    ns, nx = P.hmlfc_hierarchy_sizes(cfg.U, cfg.V, cfg.height)
    assert srv.shape == (3, ns, cfg.Ht, cfg.Ws) and x.shape == (3, nx, cfg.Ht, cfg.Ws)
    s_off = x_off = 0
    for L in range(cfg.height + 1):
        UL, VL = tree.level_dims(L)
        for c in range(3):
            for pv in range(VL):
                for pu in range(UL):
                    if L < cfg.height:
                        assert np.array_equal(srv[c, s_off + pv * UL + pu], tree.plane("srv", L, pu, pv, c)), (L, c, pu, pv)
                    if L >= 1:
                        assert np.array_equal(x[c, x_off + pv * UL + pu], tree.plane("X", L, pu, pv, c)), (L, c, pu, pv)
        if L < cfg.height:
            s_off += UL * VL
        if L >= 1:
            x_off += UL * VL
    assert s_off == ns and x_off == nx
    # path-sum identity: X_0 = X_h + sum_L SRV_L reproduces the colour-transformed input exactly
    u, v = cfg.U - 1, cfg.V // 2
    acc = x[:, nx - tree.level_dims(cfg.height)[0] * tree.level_dims(cfg.height)[1] +
            (v >> cfg.height) * tree.level_dims(cfg.height)[0] + (u >> cfg.height)].astype(np.int32)
    off = 0
    for L in range(cfg.height):
        UL, VL = tree.level_dims(L)
        acc += srv[:, off + (v >> L) * UL + (u >> L)]
        off += UL * VL
    for c in range(3):
        assert np.array_equal(acc[c], tree.plane("X", 0, u, v, c))
    tree.close()


def _cluster_pairs(UL, VL):
    """(predictive plane, reference plane) index pairs of a UL x VL level (R5: the even-even member of every
    2 x 2 cluster is the reference of the other members); plane index = pv * UL + pu."""
    return np.array([(pv * UL + pu, (pv & ~1) * UL + (pu & ~1)) for pv in range(VL) for pu in range(UL) if (pu | pv) & 1],
                    dtype=np.int32).reshape(-1, 2)


def test_hierarchy_then_search_reproduces_the_encoders_motion_decisions(P):
    """RGB light field -> hmlfc_hierarchy -> hmlfc_search on the device-resident SRV planes = the oracle encoder's (mode, dx, dy,
    SAD) of every block of every predictive plane (level 0 and 1, all channels)."""
    cfg = wl.CONFIGS["mini2"]
    lf = wl.light_field(cfg)
    tree = _tree(cfg, lf)
    srv, _ = P.hmlfc_hierarchy(torch.from_numpy(lf).cuda(), cfg.height)
    off = 0
    for L in range(cfg.height):
        UL, VL = tree.level_dims(L)
        pairs = _cluster_pairs(UL, VL)
        for c in range(3):
            planes = srv[c, off:off + UL * VL].contiguous()
            got = P.hmlfc_search(planes, torch.from_numpy(pairs).cuda(), cfg.block, cfg.window).cpu().numpy()
            for k, (pi, ri) in enumerate(pairs):
                assert np.array_equal(got[k], tree.blocks(L, int(pi) % UL, int(pi) // UL, c)[..., :4]), (L, c, pi)
        off += UL * VL
    tree.close()
