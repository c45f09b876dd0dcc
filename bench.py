#!/usr/bin/env python
"""bench.py -- HMLFC decode + fused render hot path on B200 (contract: see DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg2] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: hmlfc_render of the
configuration's view batch (ray set-up, tap enumeration, tree-walk decode with motion
re-compensation, inverse colour, quadrilinear blend, RGB8 store -- SURVEY.md 8(a) S1-S9) in ONE kernel
launch.  The second half of BASELINE.json's metric, decoded LF pixels/s (hmlfc_decode on seeded uniformly
random coordinates), is timed in the same run and reported under "decode".

Inputs: the seeded synthetic light field of the configuration (workloads/), encoded ONCE, before any timed
region.  The headline configuration (cfg2) is encoded by the oracle's encoder (oracle/streams.py, cached on disk); the
larger configurations of the `configs` object are encoded by hmlfc_encode on the GPU (the oracle would need minutes to
hours; the GPU encoder's stream is byte-identical to the oracle's on every configuration where both were run --
tests/test_gpu_encode.py).  The timed product path calls only the C-ABI library; the oracle is executed again only for
the "cpu_baseline" object and for `--impl reference`.

N > 1 (torchrun): the path shards with no exchange step -- every rank holds the stream and renders its own
batch of views (weak scaling); value = views of all ranks / max-over-ranks device time.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_FLUSH_BYTES = 512 << 20  # > 126 MB L2
RENDER_KERNEL_NAME = "render_tiles_kernel"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and clock-event reasons of one GPU while the timed region runs."""

    REASONS = (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4),
               ("hw_power_brake", 0x80), ("applications_clocks", 0x2))

    def __init__(self, index, period=0.002):
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev)
                for name, bit in self.REASONS:
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def _physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def reduce_max(x, world, device="cpu"):
    """Max over ranks of a per-rank duration (the contract's max-over-ranks timing); identity at world 1."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(x)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank_per_step, steps, world, seconds):
    """Weak scaling: every rank processes its own batch; value = units of ALL ranks / max-over-ranks time."""
    return world * units_per_rank_per_step * steps / seconds


def rank_cameras(cfg, rank):
    """The view batch of one rank: its own arc of the seeded circular camera path (no exchange between ranks)."""
    import workloads as wl

    return wl.camera_path(cfg, seed_offset=rank)


def _get_stream(name, rank, world, barrier):
    """Rank 0 encodes (oracle encoder, input preparation) into the on-disk cache; the others read it."""
    from oracle import streams

    if world == 1 or rank == 0:
        out = streams.get_stream(name)
        barrier()
        return out
    barrier()
    return streams.get_stream(name)


def _oracle_views_sample(stream, cams, W, H, budget_s, max_views):
    """Render views one by one with the oracle (all host cores) until budget_s is used."""
    t0 = time.perf_counter()
    n = 0
    while n < max_views:
        stream.render(cams[n % len(cams)][None], W, H)
        n += 1
        if time.perf_counter() - t0 >= budget_s:
            break
    return n, time.perf_counter() - t0


def run_reference(args, cfg_name):
    """--impl reference: the oracle as it stands, on the host cores; each step = a bounded sample of the batch."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as orc
    import workloads as wl
    from oracle import streams

    cfg, data, info = streams.get_stream(cfg_name)
    s = orc.Stream(data)
    cams = wl.camera_path(cfg)
    cores = os.cpu_count() or 1
    W, H = cfg.out_w, cfg.out_h
    # size the per-step sample from one view so the whole run ends within a few minutes
    t0 = time.perf_counter()
    s.render(cams[:1], W, H)
    t_view = time.perf_counter() - t0
    per_step = int(max(1, min(cfg.n_views, round(6.0 / max(t_view, 1e-3)))))
    for k in range(args.warmup):
        s.render(cams[k % len(cams)][None], W, H)
    t0 = time.perf_counter()
    for k in range(args.steps):
        idx = [(k * per_step + i) % len(cams) for i in range(per_step)]
        s.render(cams[idx], W, H)
    dt = time.perf_counter() - t0
    value = args.steps * per_step / dt
    sample = f"{per_step} of the batch's {cfg.n_views} views ({W}x{H}) per step, OpenMP over {cores} threads"
    line = {
        "impl": "reference", "metric": "rendered_views_per_s", "value": value, "unit": "views/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": _config_dict(cfg, info), "timing": {"l2": "n/a (CPU)", "clock": "host wall clock"},
        "cpu_baseline": {"value": value, "unit": "views/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "views/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def _config_dict(cfg, info):
    return {
        "workload": f"{cfg.name}: {cfg.U}x{cfg.V} views x {cfg.Ws}x{cfg.Ht} RGB8, h={cfg.height}, B={cfg.block}, W={cfg.window}; "
                    f"render {cfg.n_views} views of {cfg.out_w}x{cfg.out_h} per step on the seeded circular camera path",
        "stream_bytes": info["stream_bytes"], "stream_bpp": round(info["bpp"], 4), "psnr_db": round(info["psnr"], 3),
        "tau_res": info["tau_res"], "views_per_step": cfg.n_views, "out_w": cfg.out_w, "out_h": cfg.out_h,
        "encoder_policy": "adaptive (DESIGN.md R13: a predictive block below tau_res is dropped whole and pred is kept only where it lowers the "
                          "energy; SPEC.md's default stores a motion record for every predictive block = policy 'all')",
    }


def _timed_single(fn, steps, warmup, flush, stream):
    """Device time of `steps` calls of fn (one rank): CUDA events on the launching stream, L2 flushed before every call."""
    import torch

    for _ in range(warmup):
        flush.fill_(1)
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    torch.cuda.synchronize()
    for a, b in ev:
        flush.fill_(1)
        a.record(stream)
        fn()
        b.record(stream)
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in ev]


def measure_other_config(P, name, steps, peak, flush, stream):
    """One of the larger configurations of BASELINE.json (the `configs` object of the bench line): the configuration's light field
    (workloads/), encoded on the GPU by hmlfc_encode with the thresholds found by bisection to its PSNR target, then the same two
    timed legs as the headline -- hmlfc_render of the view batch (one launch per step) and hmlfc_decode of the random coordinates."""
    import torch

    import workloads as wl

    cfg = wl.CONFIGS[name]
    t0 = time.perf_counter()
    lf_dev = torch.from_numpy(wl.light_field(cfg)).cuda()
    t_gen = time.perf_counter() - t0
    t0 = time.perf_counter()
    data, est = P.hmlfc_encode(lf_dev, cfg.height, cfg.block, cfg.window, geometry=wl.geometry(cfg), seed=cfg.seed, target_psnr=cfg.target_psnr)
    t_enc = time.perf_counter() - t0
    del lf_dev
    P.hmlfc_encode_release_scratch()
    torch.cuda.empty_cache()
    h = P.hmlfc_load(data)
    W, H, V = cfg.out_w, cfg.out_h, cfg.n_views
    cams = torch.from_numpy(wl.camera_path(cfg)).cuda()
    out = torch.empty((V, H, W, 3), dtype=torch.uint8, device="cuda")
    n0 = P.hmlfc_launch_count(h)
    ms = _timed_single(lambda: P.hmlfc_render(h, cams, W, H, out=out, stream=stream), steps, 3, flush, stream)
    launches = P.hmlfc_launch_count(h) - n0 - 3
    fp = P.hmlfc_footprint_render(h, cams, W, H)
    kernel_ms = float(np.mean(ms))
    achieved = fp["bytes_alg"] / (kernel_ms * 1e-3) / 1e9
    coords = torch.from_numpy(wl.random_coords(cfg, cfg.n_decode)).cuda()
    dec_out = torch.empty((cfg.n_decode, 3), dtype=torch.uint8, device="cuda")
    dms = _timed_single(lambda: P.hmlfc_decode(h, coords, out=dec_out, stream=stream), max(3, min(steps, 5)), 2, flush, stream)
    fpd = P.hmlfc_footprint_decode(h, coords)
    dec_ms = float(np.mean(dms))
    dec_achieved = fpd["bytes_alg"] / (dec_ms * 1e-3) / 1e9
    res = {
        "workload": f"{cfg.name}: {cfg.U}x{cfg.V} views x {cfg.Ws}x{cfg.Ht} RGB8, h={cfg.height}, B={cfg.block}, W={cfg.window}; "
                    f"render {V} views of {W}x{H} per step on the seeded circular camera path; decode {cfg.n_decode} seeded uniformly random coordinates",
        "stream": "encoded by hmlfc_encode (GPU) with tau found by bisection to the PSNR target", "stream_bytes": len(data),
        "stream_bpp": round(8.0 * len(data) / (cfg.U * cfg.V * cfg.Ws * cfg.Ht), 4), "psnr_db": round(est["psnr"], 3), "tau_res": est["tau_res"],
        "device_bytes": int(h.info.device_bytes), "generate_s": round(t_gen, 2), "encode_s": round(t_enc, 3),
        "ms_per_step": kernel_ms, "steps": steps, "views_per_s": V / (kernel_ms * 1e-3), "output_px_per_s": V * W * H / (kernel_ms * 1e-3),
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "bytes_alg_per_launch": fp["bytes_alg"], "out_bytes": fp["out_bytes"],
                     "compressed_bytes_touched": fp["bytes_alg"] - fp["out_bytes"] - fp["in_bytes"]},
        "decode": {"value": cfg.n_decode / (dec_ms * 1e-3), "unit": "LF pixels/s", "n": cfg.n_decode, "ms_per_launch": dec_ms,
                   "roofline": {"bound": "hbm", "achieved": dec_achieved, "peak": peak, "unit": "GB/s", "frac": dec_achieved / peak,
                                "bytes_alg_per_launch": fpd["bytes_alg"]}},
    }
    P.hmlfc_free(h)
    del coords, dec_out, out, cams, data
    torch.cuda.empty_cache()
    return res


def measure_extra_stream(P, cfg_name, kind, tau_res, steps, flush, stream):
    """The rows of SURVEY 8(f) beyond the headline stream: a chroma-subsampled (R18) or a half-pel motion-compensated (R28)
    stream (both: instantiations of the fast kernels, no block records) of the headline configuration's light field, encoded by the ORACLE (hmlfc_encode does
    neither) at the headline stream's threshold; the same timed legs, and a parity spot check against the oracle."""
    import torch

    import oracle as orc
    import workloads as wl

    cfg = wl.CONFIGS[cfg_name]
    lf = wl.light_field(cfg)
    window = min(cfg.window, 4) if kind == "halfpel" else cfg.window  # the oracle's half-pel search is exhaustive over (4W + 1)^2 interpolated candidates
    p = orc.make_params(cfg.U, cfg.V, cfg.Ws, cfg.Ht, cfg.height, cfg.block, window, tau_res // 2, tau_res, geometry=wl.geometry(cfg),
                        seed=cfg.seed, chroma=1 if kind == "chroma" else 0, subpel=1 if kind == "halfpel" else 0)
    t0 = time.perf_counter()
    tree = orc.Tree(lf, p)
    data = tree.serialize()
    tree.close()
    t_enc = time.perf_counter() - t0
    s = orc.Stream(data)
    h = P.hmlfc_load(data)
    W, H, V = cfg.out_w, cfg.out_h, cfg.n_views
    cams_np = wl.camera_path(cfg)
    cams = torch.from_numpy(cams_np).cuda()
    out = torch.empty((V, H, W, 3), dtype=torch.uint8, device="cuda")
    ms = _timed_single(lambda: P.hmlfc_render(h, cams, W, H, out=out, stream=stream), steps, 2, flush, stream)
    n = min(cfg.n_decode, 2_000_000)
    coords_np = wl.random_coords(cfg, n)
    coords = torch.from_numpy(coords_np).cuda()
    dec_out = torch.empty((n, 3), dtype=torch.uint8, device="cuda")
    dms = _timed_single(lambda: P.hmlfc_decode(h, coords, out=dec_out, stream=stream), steps, 2, flush, stream)
    views = torch.from_numpy(np.array([(u, v) for v in range(cfg.V) for u in range(cfg.U)], dtype=np.int32)).cuda()
    vms = _timed_single(lambda: P.hmlfc_decode_views(h, views, stream=stream), max(2, steps // 2), 1, flush, stream)
    # parity: sampled coordinates bit-exact, one rendered view within 1 LSB
    k = 20_000
    exact = bool(np.array_equal(dec_out[:k].cpu().numpy(), s.decode(coords_np[:k])))
    ref = s.render(cams_np[:1], W, H)
    d = np.abs(out[:1].cpu().numpy().astype(np.int16) - ref.astype(np.int16))
    res = {
        "workload": f"{cfg.name} light field, oracle-encoded with {'Co / Cg at half resolution' if kind == 'chroma' else 'half-pel motion offsets'}, "
                    f"tau_res = {tau_res}, window {window}; render {V} views of {W}x{H}; decode {n} random coordinates; decode all {cfg.U * cfg.V} views",
        "kernels": ("render_tiles_kernel<kCs>, decode_rows_kernel<kCs>, decode_queue_kernel<kCs> (no block records)" if kind == "chroma" else
                    "render_tiles_kernel<kSubpel>, decode_rows_kernel<kSubpel>, decode_queue_kernel<kSubpel> (no block records)"),
        "stream_bytes": len(data), "stream_bpp": round(8.0 * len(data) / (cfg.U * cfg.V * cfg.Ws * cfg.Ht), 4),
        "psnr_db": round(float(orc.psnr(lf, s.decode_full())), 3), "oracle_encode_s": round(t_enc, 1),
        "render_ms_per_step": float(np.mean(ms)), "views_per_s": V / (float(np.mean(ms)) * 1e-3),
        "decode": {"value": n / (float(np.mean(dms)) * 1e-3), "unit": "LF pixels/s", "n": n},
        "decode_views": {"value": cfg.U * cfg.V * cfg.Ws * cfg.Ht / (float(np.mean(vms)) * 1e-3), "unit": "LF pixels/s"},
        "parity": {"decode_bit_exact_on_sample": exact, "render_max_abs_diff": int(d.max()), "render_frac_diff": float((d > 0).mean())},
    }
    P.hmlfc_free(h)
    del coords, dec_out, out, cams, views
    torch.cuda.empty_cache()
    return res


def _csrc_hash():
    """Hash of the CUDA sources the library is built from: profiles/traffic.json records it at capture time, so counters of an
    older build are recognised as stale."""
    import hashlib

    d = os.path.join(ROOT, "paper_1902_09396_b200", "csrc")
    hh = hashlib.sha1()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh", ".h")):
            with open(os.path.join(d, f), "rb") as fh:
                hh.update(f.encode() + b"\0" + fh.read())
    return hh.hexdigest()[:16]


def run_ours(args, cfg_name):
    import torch
    import torch.distributed as dist

    import paper_1902_09396_b200 as P
    import workloads as wl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the HMLFC hot path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()

    cfg, data, info = _get_stream(cfg_name, rank, world, barrier)
    h = P.hmlfc_load(data)
    if args.variant:
        P.hmlfc_set_render_variant(h, args.variant)
    if args.decode_variant:
        P.hmlfc_set_decode_variant(h, args.decode_variant)
    if args.min_level:
        P.hmlfc_set_min_level(h, args.min_level)  # progressive decoding: an extra, labelled measurement row (not the headline)
    W, H, V = cfg.out_w, cfg.out_h, cfg.n_views
    # weak scaling: every rank renders a full batch, each on its own arc of the camera circle
    cams_np = rank_cameras(cfg, rank)
    cams = torch.from_numpy(cams_np).cuda()
    out = torch.empty((V, H, W, 3), dtype=torch.uint8, device="cuda")
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def step():
        P.hmlfc_render(h, cams, W, H, out=out, stream=stream)

    def timed(fn, steps, warmup, clean_flush=False):
        # clean_flush: evict by READING the buffer, so the L2 holds clean lines when the timed kernel starts (a fill leaves up to
        # 126 MB of dirty lines whose write-back competes with an HBM-bound kernel)
        def do_flush():
            if clean_flush:
                flush.view(torch.int64).sum()
            else:
                flush.fill_(1)
        for _ in range(warmup):
            do_flush()
            fn()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        barrier()
        torch.cuda.synchronize()
        for a, b in ev:
            do_flush()              # evict the stream and the previous output from L2 (outside the events)
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        barrier()
        return [a.elapsed_time(b) for a, b in ev]

    # ---- the timed region: K steps of the fused render kernel, inputs resident in HBM
    n0 = P.hmlfc_launch_count(h)
    with ClockSampler(_physical_gpu_index(local_rank)) as clk:
        ms = timed(step, args.steps, args.warmup)
    launches = P.hmlfc_launch_count(h) - n0 - args.warmup
    total_ms = reduce_max(sum(ms), world, "cuda")
    views_per_s = whole_job_rate(V, args.steps, world, total_ms * 1e-3)

    # ---- the "grid-aligned" batch of SURVEY 8(d) D4: the same camera circle ON the camera plane (every view blends exactly 4 views)
    cams_plane = torch.from_numpy(wl.camera_path(cfg, seed_offset=rank, on_plane=True)).cuda()
    pl_ms = timed(lambda: P.hmlfc_render(h, cams_plane, W, H, out=out, stream=stream), max(3, min(args.steps, 10)), 3)
    pl_total = reduce_max(sum(pl_ms), world, "cuda")
    step()  # `out` holds the headline batch again (compared with the host entry point below)

    # ---- decode leg: seeded uniformly random LF coordinates (inputs larger than L2)
    n_dec = cfg.n_decode
    coords = torch.from_numpy(wl.random_coords(cfg, n_dec, seed_offset=rank)).cuda()
    dec_out = torch.empty((n_dec, 3), dtype=torch.uint8, device="cuda")
    dec_ms = timed(lambda: P.hmlfc_decode(h, coords, out=dec_out, stream=stream), max(3, min(args.steps, 10)), 3)
    dec_total = reduce_max(sum(dec_ms), world, "cuda")
    dec_px_per_s = whole_job_rate(n_dec, len(dec_ms), world, dec_total * 1e-3)

    # ---- dense decode: whole views (coordinates generated in the kernel), up to 2^27 light-field pixels per launch
    n_dv = max(1, min(cfg.U * cfg.V, (1 << 27) // (cfg.Ws * cfg.Ht)))
    dv_rng = np.random.Generator(np.random.PCG64(cfg.seed + 3000 + rank))
    dv_ids = dv_rng.permutation(cfg.U * cfg.V)[:n_dv]
    dv_views = torch.from_numpy(np.stack([dv_ids % cfg.U, dv_ids // cfg.U], axis=1).astype(np.int32)).cuda()
    dv_out = torch.empty((n_dv, cfg.Ht, cfg.Ws, 3), dtype=torch.uint8, device="cuda")
    dv_ms = timed(lambda: P.hmlfc_decode_views(h, dv_views, out=dv_out, stream=stream), max(3, min(args.steps, 10)), 3)
    dv_total = reduce_max(sum(dv_ms), world, "cuda")
    dv_px = n_dv * cfg.Ws * cfg.Ht
    dv_pin = torch.empty((n_dv, cfg.Ht, cfg.Ws, 3), dtype=torch.uint8).pin_memory()
    dv_views_np = dv_views.cpu().numpy()
    P.hmlfc_decode_views_host(h, dv_views_np, out=dv_pin.numpy())
    barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(3):
        P.hmlfc_decode_views_host(h, dv_views_np, out=dv_pin.numpy())
    dv_e2e_s = reduce_max(time.perf_counter() - t0, world, "cuda")
    assert torch.equal(dv_pin.cuda(), dv_out), "decode_views: host entry point and device entry point disagree"
    del dv_out, dv_pin

    # ---- random access at block granularity: as many pixels as the decode leg, in whole B x B blocks at seeded random positions
    n_blk = max(1, n_dec // (cfg.block * cfg.block))
    brng = np.random.Generator(np.random.PCG64(cfg.seed + 4000 + rank))
    blk_np = np.stack([brng.integers(0, cfg.U, n_blk), brng.integers(0, cfg.V, n_blk), brng.integers(0, cfg.Ws // cfg.block, n_blk),
                       brng.integers(0, cfg.Ht // cfg.block, n_blk)], axis=1).astype(np.int32)
    blk_d = torch.from_numpy(blk_np).cuda()
    blk_out = torch.empty((n_blk, cfg.block, cfg.block, 3), dtype=torch.uint8, device="cuda")
    blk_ms = timed(lambda: P.hmlfc_decode_blocks(h, blk_d, out=blk_out, stream=stream), max(3, min(args.steps, 10)), 3)
    blk_total = reduce_max(sum(blk_ms), world, "cuda")
    del blk_out, blk_d

    # ---- end to end through the C ABI with HOST (pinned) buffers: cameras H2D + views D2H inside the timed region
    cams_pin = torch.from_numpy(cams_np).pin_memory()
    out_pin = torch.empty((V, H, W, 3), dtype=torch.uint8).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        P.hmlfc_render_host(h, cams_pin.numpy(), W, H, out=out_pin.numpy())
    barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        P.hmlfc_render_host(h, cams_pin.numpy(), W, H, out=out_pin.numpy())   # synchronises before returning
    e2e_s = reduce_max(time.perf_counter() - t0, world, "cuda")
    e2e_views_per_s = whole_job_rate(V, e2e_steps, world, e2e_s)
    assert torch.equal(out_pin.cuda(), out), "host entry point and device entry point disagree"
    # the decode leg end to end: coordinates H2D + kernels + pixels D2H, pipelined in chunks by hmlfc_decode_host
    coords_pin = coords.cpu().pin_memory()
    dec_pin = torch.empty((n_dec, 3), dtype=torch.uint8).pin_memory()
    P.hmlfc_decode_host(h, coords_pin.numpy(), out=dec_pin.numpy())
    barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(3):
        P.hmlfc_decode_host(h, coords_pin.numpy(), out=dec_pin.numpy())
    dec_e2e_s = reduce_max(time.perf_counter() - t0, world, "cuda")
    assert torch.equal(dec_pin.cuda(), dec_out), "decode: host entry point and device entry point disagree"
    del coords_pin, dec_pin

    # ---- encoder-side leg (SURVEY 8(f) first "next" row): phase-shifted exhaustive search of one level-0 channel
    sU, sV = min(cfg.U, 16), min(cfg.V, 16)  # at most a 16 x 16 sub-grid of planes per launch
    srv = torch.from_numpy(wl.srv_like_planes(cfg, sU * sV, seed_offset=rank)).cuda()
    # (predictive plane, reference plane) pairs of the sub-grid: every plane with an odd index against the even-even plane of its
    # 2 x 2 cluster (the pairing hmlfc_encode itself uses, R5)
    pairs_np = np.array([(pv * sU + pu, (pv & ~1) * sU + (pu & ~1)) for pv in range(sV) for pu in range(sU) if (pu | pv) & 1],
                        dtype=np.int32).reshape(-1, 2)
    pairs_d = torch.from_numpy(pairs_np).cuda()
    mv_out = torch.empty((len(pairs_np), cfg.Ht // cfg.block, cfg.Ws // cfg.block, 4), dtype=torch.int32, device="cuda")
    se_ms = timed(lambda: P.hmlfc_search(srv, pairs_d, cfg.block, cfg.window, out=mv_out, stream=stream), 5, 3)
    se_total = reduce_max(sum(se_ms), world, "cuda")
    n_blocks_search = len(pairs_np) * (cfg.Ht // cfg.block) * (cfg.Ws // cfg.block)
    del srv

    # ---- encoder-side leg 2: colour transform + hierarchy build of a 16 x 16 sub-grid of views (HBM-bound streaming kernels)
    lf_d = torch.randint(0, 256, (sV, sU, cfg.Ht, cfg.Ws, 3), dtype=torch.uint8, device="cuda",
                         generator=torch.Generator(device="cuda").manual_seed(cfg.seed + rank))
    hs, hx = P.hmlfc_hierarchy(lf_d, cfg.height)
    hi_ms = timed(lambda: P.hmlfc_hierarchy(lf_d, cfg.height, srv=hs, x=hx, stream=stream), 5, 3, clean_flush=True)
    hi_total = reduce_max(sum(hi_ms), world, "cuda")
    hi_bytes = lf_d.numel() + 2 * hs.numel() + 2 * hx.numel() + 2 * (hx.numel() - 3 * hx.shape[2] * hx.shape[3] * (((sU - 1) >> cfg.height) + 1) * (((sV - 1) >> cfg.height) + 1))
    hi_px = sU * sV * cfg.Ht * cfg.Ws
    del lf_d, hs, hx

    # ---- encoder leg 3 (rank 0): the whole GPU encoder on the configuration's own light field; the stream must equal the oracle's
    encode = None
    lf_bytes = cfg.U * cfg.V * cfg.Ws * cfg.Ht * 3
    if rank == 0 and (args.encode or lf_bytes <= (256 << 20)):
        lf_dev = torch.from_numpy(wl.light_field(cfg)).cuda()
        enc_kw = dict(geometry=wl.geometry(cfg), seed=cfg.seed)
        enc_wall, enc_stats = [], None
        for k in range(4):  # first call = warm-up
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            enc_bytes, enc_stats = P.hmlfc_encode(lf_dev, cfg.height, cfg.block, cfg.window, info["tau_ref"], info["tau_res"], **enc_kw)
            if k:
                enc_wall.append(time.perf_counter() - t0)
        dev_ms = enc_stats["ms_hierarchy"] + enc_stats["ms_search"] + enc_stats["ms_classify"] + enc_stats["ms_pack"]
        encode = {
            "value": lf_bytes / 3 / float(np.mean(enc_wall)), "unit": "LF pixels/s (wall clock, stream in host memory)",
            "ms_wall": 1e3 * float(np.mean(enc_wall)), "ms_device_kernels": dev_ms,
            "ms_phases": {k: round(enc_stats[k], 4) for k in ("ms_hierarchy", "ms_search", "ms_classify", "ms_pack", "ms_assemble", "ms_wall")},
            "kernel_launches": enc_stats["kernel_launches"], "stream_equals_oracle_stream": bool(enc_bytes == data),
            "blocks": {k: enc_stats[k] for k in ("n_search_blocks", "n_pred_blocks", "n_res_blocks")},
            "oracle_encode_seconds": info.get("encode_seconds"),
            "oracle_note": "the oracle's encode of the same light field on the host cores when the cached stream was made (includes its tau bisection)",
        }
        if cfg.target_psnr is not None:  # the same with the thresholds found by bisection to the configuration's PSNR target
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            b_bytes, b_stats = P.hmlfc_encode(lf_dev, cfg.height, cfg.block, cfg.window, target_psnr=cfg.target_psnr, **enc_kw)
            encode["bisection"] = {"ms_wall": 1e3 * (time.perf_counter() - t0), "steps": b_stats["bisection_steps"], "tau_res": b_stats["tau_res"],
                                   "psnr_db": round(b_stats["psnr"], 4), "stream_equals_oracle_stream": bool(b_bytes == data)}
            del b_bytes
        del lf_dev, enc_bytes
        P.hmlfc_encode_release_scratch()

    if rank == 0:
        # ---- roofline of the dominant kernel: algorithmic bytes per launch / average launch time
        peak, peak_src = _peaks()
        fp = P.hmlfc_footprint_render(h, cams, W, H)
        kernel_ms = float(np.mean(ms))
        achieved = fp["bytes_alg"] / (kernel_ms * 1e-3) / 1e9
        fpd = P.hmlfc_footprint_decode(h, coords)
        dec_kernel_ms = float(np.mean(dec_ms))
        dec_achieved = fpd["bytes_alg"] / (dec_kernel_ms * 1e-3) / 1e9
        cap_r, cap_d = _ncu_from_profiles(cfg.name, "render"), _ncu_from_profiles(cfg.name, "decode")
        src_now = _csrc_hash()
        stale_r, stale_d = cap_r.get("csrc_sha") != src_now, cap_d.get("csrc_sha") != src_now
        roofline = {
            "bound": "hbm", "kernel": {1: "render_pixel_kernel", 4: "render_warp_kernel", 5: "render_warp_kernel"}.get(args.variant, RENDER_KERNEL_NAME), "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": cap_r.get("dram_bytes"), "peak_source": peak_src,
            "traffic_source": {"file": "profiles/traffic.json", "commit": cap_r.get("commit"), "captured_with": cap_r.get("captured_with"),
                               "csrc_sha_at_capture": cap_r.get("csrc_sha"), "csrc_sha_now": src_now, "stale": bool(stale_r)},
            "bytes_alg_per_launch": fp["bytes_alg"], "out_bytes": fp["out_bytes"],
            "compressed_bytes_touched": fp["bytes_alg"] - fp["out_bytes"] - fp["in_bytes"],
            "kernel_ms": kernel_ms, "frac_of_8TBs": achieved / 8000.0,
            "note": "achieved = algorithmic bytes / launch time.  The output (out_bytes) is WRITTEN inside the timed region but, where it fits the "
                    "126 MB L2 beside the stream traffic, most of it is still in the L2 when the kernel ends: its write-back to HBM happens during "
                    "the next L2 flush, outside the events (the ncu capture's dram__bytes_write shows how much left the L2 in the launch).",
        }
        decode = {
            "value": dec_px_per_s, "unit": "LF pixels/s", "n": n_dec, "ms_per_launch": dec_kernel_ms,
            "e2e": {"value": whole_job_rate(n_dec, 3, world, dec_e2e_s), "unit": "LF pixels/s", "h2d_bytes_per_step": 16 * n_dec,
                    "d2h_bytes_per_step": 3 * n_dec, "steps": 3},
            "roofline": {"bound": "hbm", "kernel": {1: "decode_kernel", 2: "decode_queue_kernel", 3: "decode_queue_kernel"}.get(args.decode_variant, "decode_brec_kernel"), "achieved": dec_achieved, "peak": peak, "unit": "GB/s",
                         "frac": dec_achieved / peak, "bytes_alg_per_launch": fpd["bytes_alg"],
                         "traffic": cap_d.get("dram_bytes"),
                         "traffic_source": {"file": "profiles/traffic.json", "commit": cap_d.get("commit"), "captured_with": cap_d.get("captured_with"),
                                            "csrc_sha_at_capture": cap_d.get("csrc_sha"), "stale": bool(stale_d)}},
        }
        clocks = clk.summary()
        # the bound that binds hmlfc_decode on an L2-resident stream: random 32-byte sector gathers served by the L2
        dsec = cap_d.get("l2_read_sectors")
        gpeak = _ncu_top("gather_peak").get("l2_g_sectors_per_s")
        if dsec and gpeak and not stale_d and info["stream_bytes"] < (96 << 20):
            decode["roofline"]["gather"] = {"bound": "l2-sector-gather", "achieved": dsec / (dec_kernel_ms * 1e-3) / 1e9, "peak": gpeak,
                                            "unit": "G sectors/s", "frac": dsec / (dec_kernel_ms * 1e-3) / 1e9 / gpeak, "sectors_per_launch": dsec,
                                            "source": "lts__t_sectors_srcunit_tex_op_read.sum of the committed ncu capture; the peak is a builder-measured "
                                                      "denominator (random one-sector-per-lane gathers, profiles/r01_gather_probe.md), NOT in MEASURED_PEAKS.json"}
        # the issue-slot views divide counters of the committed capture by the live launch time: only when that capture is of THIS build
        roofline["alu"] = None if stale_r else _alu_view(cap_r.get("warp_inst"), kernel_ms, clocks.get("sm_mhz"))
        decode["roofline"]["alu"] = None if stale_d else _alu_view(cap_d.get("warp_inst"), dec_kernel_ms, clocks.get("sm_mhz"))
        # search: 2 exact fp32 adds per sample, mode and offset (Eqs. 1-2): a plain-ALU bound, 128 FP32 lanes per SM
        nd2 = (2 * cfg.window + 1) ** 2
        se_adds = n_blocks_search * nd2 * cfg.block * cfg.block * 2 * 2
        se_kernel_ms = float(np.mean(se_ms))
        se_peak = 148 * 128 * (clocks.get("sm_mhz") or 1965.0) * 1e6
        search = {
            "value": whole_job_rate(n_blocks_search, len(se_ms), world, se_total * 1e-3), "unit": "blocks/s",
            "blocks_per_launch": n_blocks_search, "pairs": int(len(pairs_np)), "ms_per_launch": se_kernel_ms,
            "workload": f"level-0 planes of one channel ({sU}x{sV} x {cfg.Ws}x{cfg.Ht}, SRV-like synthetic int16), B={cfg.block}, W={cfg.window}",
            "roofline": {"bound": "alu", "kernel": "search4_kernel", "achieved": se_adds / (se_kernel_ms * 1e-3) / 1e12,
                         "peak": se_peak / 1e12, "unit": "T fp32 add/s", "frac": se_adds / (se_kernel_ms * 1e-3) / se_peak,
                         "peak_source": "148 SMs x 128 FP32 lanes x SM clock (DESIGN.md 9.6)"},
        }
        # hierarchy: every input sample read once, every output sample written once, X_1 .. X_{h-1} read once more
        hi_kernel_ms = float(np.mean(hi_ms))
        hierarchy = {
            "value": whole_job_rate(hi_px, len(hi_ms), world, hi_total * 1e-3), "unit": "LF pixels/s", "ms_per_call": hi_kernel_ms,
            "workload": f"{sU}x{sV} views x {cfg.Ws}x{cfg.Ht} RGB8 (uniform random bytes), height {cfg.height}: {cfg.height} kernel launches per call",
            "roofline": {"bound": "hbm", "kernel": "level0_kernel + levelL_kernel", "achieved": hi_bytes / (hi_kernel_ms * 1e-3) / 1e9,
                         "peak": peak, "unit": "GB/s", "frac": hi_bytes / (hi_kernel_ms * 1e-3) / 1e9 / peak, "bytes_alg_per_call": int(hi_bytes)},
        }
        cpu = None  # the oracle is timed beside the GPU on rank 0 at N = 1 only (other ranks would idle at the next barrier)
        if world == 1:
            # ---- the oracle timed beside it, on a bounded sample of the same batch
            import oracle as orc

            s = orc.Stream(data)
            if args.min_level:
                s.set_min_level(args.min_level)
            cores = os.cpu_count() or 1
            n_cpu, cpu_s = _oracle_views_sample(s, cams_np, W, H, args.cpu_budget, V)
            cpu = {"value": n_cpu / cpu_s, "unit": "views/s", "cores": cores, "kind": "oracle",
                   "sample": f"{n_cpu} of the batch's {V} views ({W}x{H}), one at a time, OpenMP over {cores} threads, {cpu_s:.1f} s"}
            # the oracle's random-access decoder on a sample of the same coordinate list: all cores, then one thread
            n_s = min(n_dec, 2_000_000)
            sample_coords = coords[:n_s].cpu().numpy()
            t0 = time.perf_counter()
            s.decode(sample_coords)
            t_all = time.perf_counter() - t0
            n_1 = max(1, n_s // 16)
            t0 = time.perf_counter()
            s.decode(sample_coords[:n_1], nthreads=1)
            t_one = time.perf_counter() - t0
            decode["cpu_baseline"] = {"value": n_s / t_all, "unit": "LF pixels/s", "cores": cores, "kind": "oracle",
                                      "sample": f"the first {n_s} of the {n_dec} coordinates, OpenMP over {cores} threads, {t_all:.2f} s",
                                      "single_thread": {"value": n_1 / t_one, "sample": f"the first {n_1} coordinates, {t_one:.2f} s"}}
            t0 = time.perf_counter()
            s.render(cams_np[:1], W, H, nthreads=1)
            cpu["single_thread"] = {"value": 1.0 / (time.perf_counter() - t0), "sample": f"1 view ({W}x{H}), one thread"}

        others = None
        if world == 1 and args.configs and args.configs != "none":
            # ---- BASELINE.json's larger configurations (north_star: "on all five configs ... on the largest config"), GPU-encoded
            others = {}
            for name in [c for c in args.configs.split(",") if c and c != cfg.name]:
                others[name] = measure_other_config(P, name, max(3, min(args.steps, 10)), peak, flush, stream)

        extras = None
        if world == 1 and args.extras and args.extras != "none":
            # ---- optional (minutes of oracle encoding): the 8(f) rows that so far have only the per-sample CUDA path
            extras = {kind: measure_extra_stream(P, cfg.name, kind, int(info["tau_res"]), max(3, min(args.steps, 5)), flush, stream)
                      for kind in args.extras.split(",") if kind in ("chroma", "halfpel")}

        line = {
            "metric": "rendered_views_per_s", "value": views_per_s, "unit": "views/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": _config_dict(cfg, info),
            "timing": {"l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB fill, outside the events)",
                       "clock": "CUDA events on the launching stream, max over ranks"},
            "e2e": {"value": e2e_views_per_s, "unit": "views/s", "h2d_bytes_per_step": int(cams_np.nbytes),
                    "d2h_bytes_per_step": int(out_pin.numel()), "steps": e2e_steps},
            "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu, "on_plane_batch": {"value": whole_job_rate(V, len(pl_ms), world, pl_total * 1e-3), "unit": "views/s", "ms_per_step": float(np.mean(pl_ms)),
                               "workload": "the same camera circle on the camera plane z = 0 (SURVEY 8(d) D4: every view blends exactly 4 light-field views)"},
            "decode_views": {"value": whole_job_rate(dv_px, len(dv_ms), world, dv_total * 1e-3), "unit": "LF pixels/s", "n_views": int(n_dv),
                             "pixels_per_launch": int(dv_px), "ms_per_launch": float(np.mean(dv_ms)),
                             "roofline": {"bound": "hbm", "kernel": "decode_rows_kernel" if cfg.block == 4 else "decode_queue_kernel<dense>",
                                          "achieved": (3 * dv_px + 8 * n_dv + info["stream_bytes"]) / (float(np.mean(dv_ms)) * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                                          "frac": (3 * dv_px + 8 * n_dv + info["stream_bytes"]) / (float(np.mean(dv_ms)) * 1e-3) / 1e9 / peak,
                                          "bytes_alg_per_launch": int(3 * dv_px + 8 * n_dv + info["stream_bytes"]),
                                          "note": "algorithmic bytes = output + view list + the whole compressed stream once (exact when every view is decoded, else an upper bound)"},
                             "e2e": {"value": whole_job_rate(dv_px, 3, world, dv_e2e_s), "unit": "LF pixels/s", "h2d_bytes_per_step": 8 * int(n_dv),
                                     "d2h_bytes_per_step": 3 * int(dv_px), "steps": 3},
                             "workload": "hmlfc_decode_views: every pixel of a seeded random set of whole views (coordinates generated in the kernel)"},
            "decode_blocks": {"value": whole_job_rate(n_blk * cfg.block * cfg.block, len(blk_ms), world, blk_total * 1e-3), "unit": "LF pixels/s",
                              "blocks_per_launch": int(n_blk), "ms_per_launch": float(np.mean(blk_ms)),
                              "workload": f"hmlfc_decode_blocks: {n_blk} whole {cfg.block} x {cfg.block} blocks at seeded uniformly random (u, v, bx, by)"},
            "decode": decode, "search": search, "hierarchy": hierarchy, "encode": encode, "configs": others, "extras": extras,
            "output_px_per_s": views_per_s * W * H, "clocks": clocks,
            "device_bytes": int(h.info.device_bytes),
            "min_level": args.min_level,
            "paper_context": "~200 fps at 512x512 on a GTX-980, Lego Knights (PAPER.md:409): another machine and light field, not the target",
        }
        print(json.dumps(line), flush=True)
    P.hmlfc_free(h)
    if world > 1:
        dist.destroy_process_group()


def _ncu_from_profiles(cfg_name, which):
    """Per-launch counters of the committed `ncu --set full` capture of this configuration (profiles/traffic.json, written
    from profiles/*.md): {"dram_bytes": dram__bytes_read.sum + dram__bytes_write.sum, "warp_inst": smsp__inst_executed.sum}
    or {} when there is no capture for the configuration."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        try:
            with open(path) as fh:
                return json.load(fh).get(cfg_name, {}).get(which, {}) or {}
        except Exception:
            return {}
    return {}


def _ncu_top(key):
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(path) as fh:
            return json.load(fh).get(key, {}) or {}
    except Exception:
        return {}


def _alu_view(warp_inst, kernel_ms, sm_mhz, n_sms=148):
    """Issue-slot view of a kernel: executed warp-instructions per second against n_sms x 4 schedulers x SM clock."""
    if not warp_inst or not sm_mhz:
        return None
    peak = n_sms * 4 * sm_mhz * 1e6
    achieved = warp_inst / (kernel_ms * 1e-3)
    return {"bound": "alu", "achieved": achieved / 1e9, "peak": peak / 1e9, "unit": "G warp-instr/s", "frac": achieved / peak,
            "warp_inst_per_launch": warp_inst, "source": "smsp__inst_executed.sum of the committed ncu capture (profiles/)"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg2")
    ap.add_argument("--variant", type=int, default=0, help="render kernel: 0 auto (= 6 cta), 1 pixel, 2 tiled, 3 blocks, 4/5 warp (A/B only)")
    ap.add_argument("--decode-variant", type=int, default=0, help="decode kernel: 0 auto (= 2 warp-cooperative), 1 thread per coordinate")
    ap.add_argument("--min-level", type=int, default=0, help="progressive decoding: sum only the levels >= this one (0 = full quality)")
    ap.add_argument("--encode", action="store_true", help="run the GPU encoder leg also on configurations whose light field exceeds 256 MB")
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--extras", default="none", help="comma list of chroma, halfpel: also measure an oracle-encoded chroma-subsampled / half-pel stream "
                                                       "of the headline light field (per-sample kernels; adds minutes of CPU encoding; off by default)")
    ap.add_argument("--configs", default="cfg3,cfg4,cfg5", help="other BASELINE.json configurations measured after the headline (GPU-encoded "
                    "streams; N = 1 only); 'none' to skip")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args, args.config)
    else:
        run_ours(args, args.config)


if __name__ == "__main__":
    main()
