"""World-size-2 `gloo` test of the N > 1 host logic of bench.py, on CPU.

The path shards with no exchange step: every rank holds the whole (read-only) stream and processes its own units; the
only collectives are the barrier and the max-over-ranks of the timing.  Here two CPU processes run that logic with
the ORACLE standing in for the kernels (this is a test of sharding, rendezvous and reduction, not of the CUDA path).
"""
import os
import socket
import sys
import tempfile

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
torch = pytest.importorskip("torch")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, cache, outdir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      HMLFC_CACHE=cache, OMP_NUM_THREADS="2")
    import torch.distributed as dist

    import bench
    import oracle as orc
    import workloads as wl

    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank 0 encodes into the shared cache, the others read the same bytes after the barrier
    cfg, data, info = bench._get_stream("cfg1_lossy", rank, world, dist.barrier)
    s = orc.Stream(data)
    # weak scaling of the render leg: every rank renders its own batch on its own arc of the camera path
    cams = bench.rank_cameras(cfg, rank)
    views = s.render(cams, cfg.out_w, cfg.out_h)
    # strong split of one coordinate list (hmlfc_decode shards the same way): contiguous, disjoint, complete
    coords = wl.random_coords(cfg, 10_001)
    lo, hi = wl.shard(len(coords), rank, world)
    part = s.decode(coords[lo:hi])
    # max-over-ranks timing: rank r pretends to have taken (r + 1) * 10 ms
    t_max = bench.reduce_max((rank + 1) * 10.0, world, "cpu")
    value = bench.whole_job_rate(cfg.n_views, 5, world, t_max * 1e-3)
    np.savez(os.path.join(outdir, f"rank{rank}.npz"), stream=np.frombuffer(data, np.uint8), cams=cams, views=views,
             lo=lo, hi=hi, part=part, t_max=t_max, value=value, cached=info["cached"])
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_without_exchange_and_reduce_the_timing():
    import torch.multiprocessing as mp

    import oracle as orc
    import workloads as wl

    world = 2
    with tempfile.TemporaryDirectory() as cache, tempfile.TemporaryDirectory() as outdir:
        mp.spawn(_worker, args=(world, _free_port(), cache, outdir), nprocs=world, join=True)
        r = [np.load(os.path.join(outdir, f"rank{k}.npz")) for k in range(world)]
    # one encode (rank 0), identical stream bytes on every rank
    assert not bool(r[0]["cached"]) and bool(r[1]["cached"])
    assert np.array_equal(r[0]["stream"], r[1]["stream"])
    # different, seeded camera arcs per rank; each rank's views are what a single process renders for those cameras
    cfg = wl.CONFIGS["cfg1_lossy"]
    s = orc.Stream(r[0]["stream"].tobytes())
    assert not np.array_equal(r[0]["cams"], r[1]["cams"])
    for k in range(world):
        assert np.array_equal(r[k]["cams"], wl.camera_path(cfg, seed_offset=k))
        assert np.array_equal(r[k]["views"], s.render(r[k]["cams"], cfg.out_w, cfg.out_h))
    # the coordinate shards tile [0, n) and their concatenation is the single-process decode
    coords = wl.random_coords(cfg, 10_001)
    assert int(r[0]["lo"]) == 0 and int(r[0]["hi"]) == int(r[1]["lo"]) and int(r[1]["hi"]) == len(coords)
    assert np.array_equal(np.concatenate([r[0]["part"], r[1]["part"]]), s.decode(coords))
    # timing = max over ranks on every rank; value = units of all ranks / that time
    for k in range(world):
        assert float(r[k]["t_max"]) == 20.0
        assert abs(float(r[k]["value"]) - world * cfg.n_views * 5 / 20e-3) < 1e-9


def test_shard_covers_everything_for_any_world_size():
    import workloads as wl

    for n in (0, 1, 7, 64, 10 ** 8):
        for world in (1, 2, 3, 8):
            edges = [wl.shard(n, k, world) for k in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[k][1] == edges[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
