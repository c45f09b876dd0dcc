"""Encoded streams of the workload configurations, made by the ORACLE encoder and cached on disk.

TEST INFRASTRUCTURE.  The compressed streams that tests, smoke() and bench.py's headline feed to the
CUDA path are manufactured here, by the oracle's encoder, before any timed region, so that no
input of a parity test comes from the CUDA path (the GPU encoder hmlfc_encode exists as well and
is checked byte for byte against these streams).  Nothing in this module is ever called from
paper_1902_09396_b200/.

Cache: $HMLFC_CACHE or /tmp/hmlfc_cache, keyed by the configuration and a hash of the oracle and
generator sources, so a stale stream is never reused after the encoder changes.
"""
import hashlib
import json
import os
import time

import numpy as np

import workloads as wl

from . import Stream, encode, make_params, psnr  # noqa: F401

_HERE = os.path.dirname(os.path.abspath(__file__))


def _source_hash() -> str:
    h = hashlib.sha1()
    # the encoder side only: decode.c / render.c do not influence the bytes of a stream
    files = [os.path.join(_HERE, f) for f in sorted(os.listdir(_HERE)) if f.endswith((".c", ".h")) and f not in ("decode.c", "render.c")]
    files += [os.path.join(os.path.dirname(wl.__file__), f) for f in ("lfgen.c", "__init__.py")]
    for f in files:
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def cache_dir() -> str:
    d = os.environ.get("HMLFC_CACHE", "/tmp/hmlfc_cache")
    os.makedirs(d, exist_ok=True)
    return d


def get_stream(name: str, use_cache: bool = True, keep_lf: bool = False):
    """Returns (cfg, stream_bytes, info).  info: psnr, bpp, tau_res, tau_ref, stream_bytes,
    encode_seconds, generate_seconds, cached; plus 'lf' when keep_lf."""
    cfg = wl.CONFIGS[name]
    key = hashlib.sha1((repr(cfg) + _source_hash()).encode()).hexdigest()[:16]
    base = os.path.join(cache_dir(), f"{name}_{key}")
    if use_cache and not keep_lf and os.path.exists(base + ".hmlfc") and os.path.exists(base + ".json"):
        with open(base + ".hmlfc", "rb") as fh:
            data = fh.read()
        with open(base + ".json") as fh:
            info = json.load(fh)
        info["cached"] = True
        return cfg, data, info
    t0 = time.time()
    lf = wl.light_field(cfg)
    t1 = time.time()
    p = make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, cfg.window, cfg.tau_res // 2, cfg.tau_res,
                    geometry=wl.geometry(cfg), seed=cfg.seed)
    data, info, tree = encode(lf, p, cfg.target_psnr)
    tree.close()
    info = {k: (float(v) if isinstance(v, (float, np.floating)) else int(v)) for k, v in info.items()}
    info["generate_seconds"], info["encode_seconds"], info["cached"] = t1 - t0, time.time() - t1, False
    if use_cache:
        with open(base + ".hmlfc.tmp", "wb") as fh:
            fh.write(data)
        os.replace(base + ".hmlfc.tmp", base + ".hmlfc")
        with open(base + ".json", "w") as fh:
            json.dump(info, fh)
    if keep_lf:
        info["lf"] = lf
    return cfg, data, info
