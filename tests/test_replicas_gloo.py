"""N > 1 is "replicas only" (DESIGN.md §8 / SURVEY.md §8(e)): bench.py runs one independent replica per rank and
combines only timings.  This CPU test runs the rank logic with world_size 2 over gloo: distinct seeds per rank, MAX
reduction of the per-rank time, aggregate value = world * atoms * steps / max time, rank 0 reports."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import gen
    import bench
    # each rank draws its own replica (bench.py's seed rule)
    coord, types, box = gen.make_system("W192", seed=gen.SEED_BASE + gen.CONFIGS["W192"].config_id + 7919 * rank)
    fake_ms = 10.0 * (rank + 1)                                   # rank 1 is the slow one
    t = torch.tensor([fake_ms, 2 * fake_ms], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.barrier()
    steps, n = 4, coord.shape[0]
    value = world * n * steps / (float(t[0]) * 1e-3)
    flops = bench.algorithmic_flops(gen.weights.MODELS["W192"], n, 16000)
    q.put((rank, float(coord.sum()), float(t[0]), value, flops["pass1"] > 0))
    dist.destroy_process_group()


def test_world_size_2_replicas_over_gloo():
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
    (r0, s0, t0, v0, ok0), (r1, s1, t1, v1, ok1) = res
    assert s0 != s1                       # different replicas
    assert t0 == t1 == 20.0               # max over ranks
    assert v0 == v1 == 2 * 192 * 4 / 20e-3
    assert ok0 and ok1


def test_algorithmic_flops_match_the_survey_table():
    """12,550 / 20,544 embedding GEMM flop per neighbour and direction; 998,880 / 1,213,920 fitting
    flop per atom and direction."""
    sys.path.insert(0, ROOT)
    import bench
    from gen.weights import MODELS
    for name, gemm, fit in (("W24k", 12550, 998880), ("Cu32k", 20544, 1213920)):
        spec = MODELS[name]
        s1 = spec.emb_s1
        assert 2 * (s1 + 2 * s1 * s1 + 8 * s1 * s1) == gemm
        assert 2 * (spec.dim_descrpt * 240 + 2 * 240 * 240 + 240) == fit
        f = bench.algorithmic_flops(spec, 1, 1)
        assert f["pass1"] > gemm and f["pass2"] > gemm and f["fit"] > 2 * fit
