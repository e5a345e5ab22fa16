"""bench.py's N > 1 path on CPU: world-size-2 gloo.  Every rank takes its own scan (same recipe, seed + 1000 rank),
the elapsed time is the MAX over ranks and the value is the whole-job aggregate."""
import argparse
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import bench
    import synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    args = argparse.Namespace(config=1, grid=4, iters=0)
    cfg, iters = bench.workload(args, rank)
    pos = synth.positions(cfg)
    obj = synth.true_object(cfg)
    ms = bench.max_over_ranks(10.0 * (rank + 1), dist, torch.device("cpu"))
    value = bench.job_value(world, cfg.K, iters, 3, ms)
    # every rank must see the same aggregate
    t = torch.tensor([value], dtype=torch.float64)
    lo, hi = t.clone(), t.clone()
    dist.all_reduce(lo, op=dist.ReduceOp.MIN)
    dist.all_reduce(hi, op=dist.ReduceOp.MAX)
    out[rank] = dict(seed=cfg.seed, K=cfg.K, iters=iters, ms=ms, value=value, same=bool(lo.item() == hi.item()),
                     obj00=complex(obj[0, 0]), pos_sum=int(pos.sum()))
    dist.destroy_process_group()


def test_two_ranks_weak_scaling_logic():
    world = 2
    port = _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r1["seed"] == r0["seed"] + 1000          # independent scans
    assert r0["obj00"] != r1["obj00"]                # different objects
    assert r0["pos_sum"] == r1["pos_sum"]            # config 1 has no jitter: same geometry
    assert r0["K"] == r1["K"] == 16 and r0["iters"] == 100
    assert r0["ms"] == r1["ms"] == 20.0              # max over ranks
    assert r0["same"] and r1["same"]
    assert np.isclose(r0["value"], 2 * 16 * 100 * 3 / 20e-3)
