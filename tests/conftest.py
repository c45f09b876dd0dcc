import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


_cache = {}


def encoded(name):
    """(cfg, lf, stream_bytes, info, oracle Stream) of a workloads config, encoded once per session
    by the ORACLE encoder (the CUDA path never produces streams or expected values)."""
    if name in _cache:
        return _cache[name]
    import oracle as orc
    import workloads as wl

    cfg = wl.CONFIGS[name]
    lf = wl.light_field(cfg)
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, cfg.tau_res // 2, cfg.tau_res,
                        geometry=wl.geometry(cfg), seed=cfg.seed)
    data, info, tree = orc.encode(lf, p, cfg.target_psnr)
    info["p1"] = tree.reconstruct()
    tree.close()
    _cache[name] = (cfg, lf, data, info, orc.Stream(data))
    return _cache[name]


@pytest.fixture(scope="session")
def enc():
    return encoded


def random_lf(rng, U, V, Ws, Ht, smooth=True):
    """Small random RGB8 light field with inter-view coherence (shifted copies of one noise image + noise)."""
    base = rng.integers(0, 256, (Ht + 16, Ws + 16, 3)).astype(np.float64)
    if smooth:
        for _ in range(2):
            base = (base + np.roll(base, 1, 0) + np.roll(base, 1, 1) + np.roll(base, (1, 1), (0, 1))) / 4.0
    lf = np.empty((V, U, Ht, Ws, 3), dtype=np.uint8)
    for v in range(V):
        for u in range(U):
            dx, dy = (u * 3) % 8, (v * 2) % 8
            img = base[dy:dy + Ht, dx:dx + Ws] + rng.normal(0, 2.0, (Ht, Ws, 3))
            lf[v, u] = np.clip(np.rint(img), 0, 255).astype(np.uint8)
    return lf
