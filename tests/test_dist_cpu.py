"""World-size-2 gloo test (CPU) of the replica-parallel host logic used by bench.py --gpus N."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_05650_b200 import dist as gdist


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    frames = gdist.frame_shard(7, rank, world)
    ms = 10.0 if rank == 0 else 25.0                      # rank 1 is the slow replica
    units = 1_000_000 * len(frames)
    thr = gdist.job_throughput(units, ms)
    out.put((rank, list(frames), gdist.max_over_ranks(ms), gdist.sum_over_ranks(len(frames)), thr))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_sharding_and_timing_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    frames = [f for _, fr, *_ in res for f in fr]
    assert sorted(frames) == list(range(7))                      # every frame exactly once
    assert [len(r[1]) for r in res] == [4, 3]
    for _, _, mx, tot, thr in res:
        assert mx == 25.0 and tot == 7.0
        assert abs(thr - 7_000_000 / 0.025) < 1e-6


def test_frame_shard_properties():
    for n in (0, 1, 5, 8, 300):
        for world in (1, 2, 3, 8):
            parts = [gdist.frame_shard(n, r, world) for r in range(world)]
            assert sorted(f for p in parts for f in p) == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1


def test_single_process_passthrough():
    assert gdist.max_over_ranks(3.5) == 3.5 and gdist.sum_over_ranks(2.0) == 2.0
